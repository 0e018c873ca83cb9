"""GPU test of nqs_weighted_stats_static, the one entry point of libnqs that allocates no device memory.

It exists for callers that cannot let a library call cudaMalloc: a VMC loop whose framework allocator already owns the
whole card, a multi-stream loop that cannot take cudaMalloc's device-wide synchronisation, a process on a fixed memory
budget (include/nqs.h).  Its scratch is a fixed array inside the library that every call on the device shares and
that keeps the previous call's contents, so the thing to check is exactly: two calls in a row, of different sizes,
each equal to what the existing path (the statistics nqs_local_energy returns, accumulated in its handle workspace)
gives for the same rows — at the tolerance the parity tests use for those statistics (rtol 1e-9, fp64 sums in a
different order).

The file sorts last on purpose (pytest -x stops at the first failure; nothing should hide behind this one) and builds
its own inputs, so it passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import paper_2208_05637_b200 as nqs
from paper_2208_05637_b200 import workloads as wl

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _dev_u64(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int64)).to(DEV)


def test_static_scratch_stats_match_the_workspace_path_on_two_calls_in_a_row():
    torch.cuda.set_device(0)
    w = wl.WORKLOADS[1]                                   # 8 qubits, 361 terms: E_loc of 10^4 rows takes milliseconds
    h, g = wl.make_integrals(w.n_spatial, w.seed_integrals)
    x, z, c = wl.jw_pauli_terms(h, g)
    H = nqs.ham_compile_packed(w.n_qubits, x, z, c)
    M = nqs.made_create(wl.make_made_params(w.n_qubits, w.hidden, w.seed_weights))
    B1, B2 = 10_000, 4_097                                # 5 CTAs with a ragged tail, then 3 CTAs (2 full + 1 row)
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, B1, 1024, w.seed_samples, False)
    xs, cn = _dev_u64(samples), torch.from_numpy(counts).to(DEV)

    # existing path: E_loc and its statistics (device accumulator in the handle's workspace, read back to the host)
    e1, ref1 = nqs.local_energy(H, M, xs, cn, minibatch=4096)
    e2, ref2 = nqs.local_energy(H, M, xs[:B2].contiguous(), None)
    assert ref1[0] == counts.sum() and ref2[0] == B2

    # every buffer of the new entry point is the caller's and exists before the calls
    out1 = torch.full((4,), float("nan"), dtype=torch.float64, device=DEV)
    out2 = torch.full((4,), float("nan"), dtype=torch.float64, device=DEV)
    nqs.weighted_stats_static(e1, cn, out1)               # first call on this device: also looks the scratch up
    nqs.weighted_stats_static(e2, None, out2)             # second call, same stream: reuses the scratch, fewer CTAs
    torch.cuda.synchronize()
    np.testing.assert_allclose(out1.cpu().numpy(), ref1[:4], rtol=1e-9)
    np.testing.assert_allclose(out2.cpu().numpy(), ref2[:4], rtol=1e-9)

    # and the first shape once more: the result is a fixed-order sum, so it repeats bit for bit
    out3 = torch.empty(4, dtype=torch.float64, device=DEV)
    nqs.weighted_stats_static(e1, cn, out3)
    assert out3.cpu().numpy().tobytes() == out1.cpu().numpy().tobytes()

    # B = 0 writes zeros; a size beyond the fixed scratch is refused before anything is launched
    nqs.weighted_stats_static(e1[:0], None, out3)
    assert (out3.cpu().numpy() == 0).all()
    rc = nqs.lib().nqs_weighted_stats_static(e1.data_ptr(), None, nqs.STATS_STATIC_MAX_ROWS + 1, out3.data_ptr(), None)
    assert rc == -2 and b"range" in nqs.lib().nqs_strerror(rc)
