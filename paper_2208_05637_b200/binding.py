"""Thin ctypes binding over libnqs.so (include/nqs.h).  Argument marshalling only: every step of the hot
path runs inside the library's CUDA kernels.  There is no CPU fallback — if the library cannot be loaded,
or no sm_100 device is usable, calls raise."""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libnqs.so")

PATH_AUTO, PATH_SIMT, PATH_TC = 0, 1, 2
_lib = None

c_void_p, c_int, c_int64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64


class NqsError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: {lib().nqs_strerror(status).decode()} (status {status})")


def lib():
    """Load libnqs.so (fails loudly when the CUDA extension has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2208_05637_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        L.nqs_strerror.restype = ctypes.c_char_p
        L.nqs_strerror.argtypes = [c_int]
        L.nqs_ham_compile.argtypes = [c_int, c_int64, c_void_p, c_void_p, ctypes.POINTER(c_void_p)]
        L.nqs_ham_compile_packed.argtypes = [c_int, c_int64, c_void_p, c_void_p, c_void_p, ctypes.POINTER(c_void_p)]
        L.nqs_ham_compile_text.argtypes = [c_int, ctypes.c_char_p, ctypes.POINTER(c_void_p)]
        L.nqs_ham_info.argtypes = [c_void_p, ctypes.POINTER(c_int), ctypes.POINTER(c_int64),
                                   ctypes.POINTER(c_int64), ctypes.POINTER(ctypes.c_double)]
        L.nqs_ham_export.argtypes = [c_void_p] * 6
        L.nqs_ham_free.argtypes = [c_void_p]
        L.nqs_ham_free.restype = None
        L.nqs_made_create.argtypes = [c_int, c_int, c_int, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                                      c_void_p, ctypes.POINTER(c_void_p)]
        L.nqs_made_export_masked.argtypes = [c_void_p, c_int, c_void_p]
        L.nqs_made_free.argtypes = [c_void_p]
        L.nqs_made_path.argtypes = [c_void_p, c_int]
        L.nqs_made_tc_flops.argtypes = [c_void_p, ctypes.POINTER(c_int64), ctypes.POINTER(c_int64)]
        L.nqs_made_free.restype = None
        L.nqs_made_logpsi.argtypes = [c_void_p, c_void_p, c_int64, c_void_p, c_int, c_void_p]
        L.nqs_pauli_contract.argtypes = [c_void_p, c_void_p, c_int64, c_int64, c_int64, c_void_p, c_void_p]
        L.nqs_local_energy.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int64, c_int64, c_int,
                                       c_void_p, c_void_p, c_void_p]
        L.nqs_local_energy_host.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int64, c_int64, c_int,
                                            c_void_p, c_void_p]
        L.nqs_weighted_stats_static.argtypes = [c_void_p, c_void_p, c_int64, c_void_p, c_void_p]
        L.nqs_made_set_constraint.argtypes = [c_void_p, c_int, c_int]
        L.nqs_made_num_params.argtypes = [c_void_p, ctypes.POINTER(c_int64)]
        L.nqs_energy_grad.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int64, c_int64, c_void_p, c_void_p, c_void_p, c_void_p]
        L.nqs_made_sample.argtypes = [c_void_p, c_int64, ctypes.c_uint64, c_int, c_int, c_int64, c_void_p, c_void_p,
                                      ctypes.POINTER(c_int64), c_void_p]
        L.nqs_kernel_launch_count.restype = c_int64
        L.nqs_kernel_launch_count.argtypes = []
        L.nqs_last_chain_kernel_ms.argtypes = [c_void_p, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(c_int)]
        _lib = L
    return _lib


def _chk(status, where):
    if status != 0:
        raise NqsError(status, where)


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


class Hamiltonian:
    """nqs_ham_t handle (nqs_ham_compile / nqs_ham_compile_packed)."""

    def __init__(self, handle):
        self._h = handle
        n, K, G, s = c_int(), c_int64(), c_int64(), ctypes.c_double()
        _chk(lib().nqs_ham_info(self._h, n, K, G, s), "nqs_ham_info")
        self.n_qubits, self.K, self.G, self.sum_abs_coeff = n.value, K.value, G.value, s.value

    def export(self):
        K, G = self.K, self.G
        out = dict(flips=np.zeros((G, 2), np.uint64), offsets=np.zeros(G + 1, np.uint32),
                   zy=np.zeros((K, 2), np.uint64), ycount=np.zeros(K, np.uint8), coef=np.zeros(K, np.float32))
        _chk(lib().nqs_ham_export(self._h, out["flips"].ctypes.data, out["offsets"].ctypes.data,
                                  out["zy"].ctypes.data, out["ycount"].ctypes.data, out["coef"].ctypes.data),
             "nqs_ham_export")
        return out

    def __del__(self):
        if getattr(self, "_h", None):
            lib().nqs_ham_free(self._h)
            self._h = None


def ham_compile(codes, coeffs, n_qubits=None):
    codes = _np(codes, np.uint8)
    coeffs = _np(coeffs, np.float64)
    K = codes.shape[0]
    n = int(n_qubits if n_qubits is not None else codes.shape[1])
    h = c_void_p()
    _chk(lib().nqs_ham_compile(n, K, codes.ctypes.data, coeffs.ctypes.data, ctypes.byref(h)), "nqs_ham_compile")
    return Hamiltonian(h)


def ham_compile_text(n_qubits, text):
    """Hamiltonian from text: 'coeff IXYZ...' or 'coeff [X0 Y3 Z12]' per line (include/nqs.h)."""
    h = c_void_p()
    _chk(lib().nqs_ham_compile_text(int(n_qubits), text.encode(), ctypes.byref(h)), "nqs_ham_compile_text")
    return Hamiltonian(h)


def ham_compile_packed(n_qubits, fmask, smask, coeffs):
    fmask, smask, coeffs = _np(fmask, np.uint64), _np(smask, np.uint64), _np(coeffs, np.float64)
    h = c_void_p()
    _chk(lib().nqs_ham_compile_packed(int(n_qubits), coeffs.shape[0], fmask.ctypes.data, smask.ctypes.data,
                                      coeffs.ctypes.data, ctypes.byref(h)), "nqs_ham_compile_packed")
    return Hamiltonian(h)


class Made:
    """nqs_made_t handle (nqs_made_create)."""

    def __init__(self, handle, n, hidden, layers):
        self._h, self.n_qubits, self.hidden, self.n_hidden_layers = handle, n, hidden, layers

    def export_masked(self, layer):
        n, h, L = self.n_qubits, self.hidden, self.n_hidden_layers
        shape = (h, n) if layer == 0 else ((n, h) if layer == L else (h, h))
        out = np.zeros(shape, np.float32)
        _chk(lib().nqs_made_export_masked(self._h, layer, out.ctypes.data), "nqs_made_export_masked")
        return out

    def resolved_path(self, path=PATH_AUTO):
        r = lib().nqs_made_path(self._h, path)
        if r < 0:
            raise NqsError(r, "nqs_made_path")
        return r

    def set_constraint(self, n_up=-1, n_down=-1):
        _chk(lib().nqs_made_set_constraint(self._h, n_up, n_down), "nqs_made_set_constraint")

    def num_params(self):
        k = c_int64()
        _chk(lib().nqs_made_num_params(self._h, k), "nqs_made_num_params")
        return k.value

    def tc_flops(self):
        """(issued, dense) tensor-core flops per psi evaluation of NQS_PATH_TC (nqs_made_tc_flops)."""
        a, b = c_int64(), c_int64()
        _chk(lib().nqs_made_tc_flops(self._h, a, b), "nqs_made_tc_flops")
        return a.value, b.value

    def last_chain_kernel_ms(self):
        ms, k = ctypes.c_float(), c_int()
        _chk(lib().nqs_last_chain_kernel_ms(self._h, ms, k), "nqs_last_chain_kernel_ms")
        return ms.value, k.value

    def __del__(self):
        if getattr(self, "_h", None):
            lib().nqs_made_free(self._h)
            self._h = None


def _ptr_array(arrs):
    keep = [_np(a, np.float32) for a in arrs]
    return (c_void_p * len(keep))(*[a.ctypes.data for a in keep]), keep


def made_create(params):
    """params: any object with the fields of workloads.MadeParams."""
    n, h, L = int(params.n_qubits), int(params.hidden), int(params.n_hidden_layers)
    order = _np(params.order, np.int32) if params.order is not None else None
    deg = _np(params.deg_hidden, np.int32) if params.deg_hidden is not None else None
    w, kw = _ptr_array(params.weights)
    b, kb = _ptr_array(params.biases)
    pw, kpw = _ptr_array(params.phase_weights)
    pb, kpb = _ptr_array(params.phase_biases)
    hd = c_void_p()
    _chk(lib().nqs_made_create(n, h, L, order.ctypes.data if order is not None else None,
                               deg.ctypes.data if deg is not None else None, w, b, pw, pb, ctypes.byref(hd)),
         "nqs_made_create")
    return Made(hd, n, h, L)


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def made_logpsi(made, configs, path=PATH_AUTO, stream=None):
    """configs: torch.int64 CUDA tensor [B, 2] holding the uint64 bit patterns -> torch.float32 [B, 2]."""
    import torch
    B = configs.shape[0]
    out = torch.empty((B, 2), dtype=torch.float32, device=configs.device)
    _chk(lib().nqs_made_logpsi(made._h, configs.data_ptr(), B, out.data_ptr(), path, _stream_ptr(stream)),
         "nqs_made_logpsi")
    return out


def pauli_contract(ham, samples, g0=0, g1=None, stream=None):
    """-> torch.float32 [g1-g0, B, 2]."""
    import torch
    g1 = ham.G if g1 is None else g1
    B = samples.shape[0]
    out = torch.empty((g1 - g0, B, 2), dtype=torch.float32, device=samples.device)
    _chk(lib().nqs_pauli_contract(ham._h, samples.data_ptr(), B, g0, g1, out.data_ptr(), _stream_ptr(stream)),
         "nqs_pauli_contract")
    return out


def local_energy(ham, made, samples, counts=None, minibatch=0, path=PATH_AUTO, want_stats=True, stream=None,
                 out=None):
    """samples: torch.int64 CUDA [B, 2]; counts: torch.int64 CUDA [B] or None.
    Returns (eloc torch.float32 [B, 2], stats np.float64 [5] or None)."""
    import torch
    B = samples.shape[0]
    if out is None:
        out = torch.empty((B, 2), dtype=torch.float32, device=samples.device)
    stats = np.zeros(5, np.float64) if want_stats else None
    _chk(lib().nqs_local_energy(ham._h, made._h, samples.data_ptr(), counts.data_ptr() if counts is not None else None,
                                B, minibatch, path, out.data_ptr(), stats.ctypes.data if want_stats else None,
                                _stream_ptr(stream)), "nqs_local_energy")
    return out, stats


def local_energy_host(ham, made, samples, counts=None, minibatch=0, path=PATH_AUTO, want_stats=True, out=None):
    """Host-buffer variant: samples np.uint64 [B, 2], counts np.int64 [B] or None -> (np.float32 [B, 2], stats)."""
    samples = _np(samples, np.uint64)
    B = samples.shape[0]
    cnt = _np(counts, np.int64) if counts is not None else None
    if out is None:
        out = np.zeros((B, 2), np.float32)
    stats = np.zeros(5, np.float64) if want_stats else None
    _chk(lib().nqs_local_energy_host(ham._h, made._h, samples.ctypes.data, cnt.ctypes.data if cnt is not None else None,
                                     B, minibatch, path, out.ctypes.data, stats.ctypes.data if want_stats else None),
         "nqs_local_energy_host")
    return out, stats


STATS_STATIC_MAX_ROWS = 1 << 21


def weighted_stats_static(eloc, counts, out, stream=None):
    """nqs_weighted_stats_static: the sums of Eq. 17 for callers that cannot let the library allocate device memory
    (a framework allocator owns the card, cudaMalloc's device-wide synchronisation is unaffordable, or the process has a
    fixed memory budget).  Nothing is allocated here either: the caller brings every buffer.
    eloc torch.float32 CUDA [B, 2], counts torch.int64 CUDA [B] or None, out torch.float64 CUDA [4] (overwritten with
    sum n, sum n Re E, sum n Im E, sum n |E|^2; returned).  B <= STATS_STATIC_MAX_ROWS.  Asynchronous on the stream.
    Calls on one device share a fixed scratch array inside the library: do not let two of them overlap on the GPU, and
    make the first call on a device before any stream capture (include/nqs.h)."""
    import torch
    if not (out.is_cuda and out.dtype == torch.float64 and out.numel() >= 4 and out.is_contiguous()):
        raise ValueError("out must be a contiguous CUDA float64 tensor of at least 4 elements")
    if not (eloc.is_cuda and eloc.dtype == torch.float32 and eloc.is_contiguous()):
        raise ValueError("eloc must be a contiguous CUDA float32 tensor [B, 2]")
    if counts is not None and not (counts.is_cuda and counts.dtype == torch.int64 and counts.is_contiguous()
                                   and counts.shape[0] == eloc.shape[0]):
        raise ValueError("counts must be a contiguous CUDA int64 tensor [B]")
    _chk(lib().nqs_weighted_stats_static(eloc.data_ptr(), counts.data_ptr() if counts is not None else None,
                                         eloc.shape[0], out.data_ptr(), _stream_ptr(stream)), "nqs_weighted_stats_static")
    return out


def energy_grad(made, samples, counts, eloc, minibatch=0, want_baseline=True, stream=None, global_stats=None):
    """Gradient of Eq. 7.  samples torch.int64 CUDA [B, 2], counts torch.int64 CUDA [B] or None, eloc torch.float32 CUDA
    [B, 2] -> (grad torch.float32 [n_params], baseline complex or None)."""
    import torch
    B = samples.shape[0]
    grad = torch.empty((made.num_params(),), dtype=torch.float32, device=samples.device)
    base = np.zeros(2, np.float64) if want_baseline else None
    gs = _np(global_stats, np.float64) if global_stats is not None else None
    _chk(lib().nqs_energy_grad(made._h, samples.data_ptr(), counts.data_ptr() if counts is not None else None,
                               eloc.data_ptr(), B, minibatch, gs.ctypes.data if gs is not None else None, grad.data_ptr(),
                               base.ctypes.data if want_baseline else None, _stream_ptr(stream)), "nqs_energy_grad")
    return grad, (complex(base[0], base[1]) if want_baseline else None)


def made_sample(made, n_draws, seed, n_up=-1, n_down=-1, max_unique=0, device="cuda", stream=None):
    """Buffer / counter sampler -> (samples torch.int64 [U, 2] holding the uint64 bit patterns, counts torch.int64 [U])."""
    import torch
    cap = max_unique if 0 < max_unique < n_draws else n_draws
    samples = torch.zeros((max(cap, 1), 2), dtype=torch.int64, device=device)
    counts = torch.zeros((max(cap, 1),), dtype=torch.int64, device=device)
    nu = c_int64()
    _chk(lib().nqs_made_sample(made._h, n_draws, seed, n_up, n_down, max_unique, samples.data_ptr(), counts.data_ptr(),
                               ctypes.byref(nu), _stream_ptr(stream)), "nqs_made_sample")
    return samples[:nu.value], counts[:nu.value]


def kernel_launch_count():
    return int(lib().nqs_kernel_launch_count())
