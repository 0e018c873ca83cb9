"""ctypes wrapper around jwgen.c (fast Jordan-Wigner input generator) + mask<->code helpers.

Pure input plumbing: the Pauli list it returns is an INPUT of the hot path
(`nqs_ham_compile`), PAPER.md:36 "store the result in a string format", :154 "Operator Matrix".
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "_jwgen.so")
_lib = None


def build_jwgen(force: bool = False) -> str:
    """Compile jwgen.c -> _jwgen.so in-tree with gcc (called by __graft_entry__.build())."""
    src = os.path.join(_HERE, "jwgen.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-shared", "-fPIC", src, "-o", _SO, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build_jwgen()
        lib = ctypes.CDLL(_SO)
        lib.jw_build.restype = ctypes.c_int64
        lib.jw_build.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double,
                                 ctypes.c_int, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p,
                                 ctypes.c_void_p, ctypes.POINTER(ctypes.c_double)]
        _lib = lib
    return _lib


def jw_pauli_terms(h: np.ndarray, g: np.ndarray, tol: float = 1e-8):
    """Integrals -> (x uint64[K,2], z uint64[K,2], coeffs float64[K]).

    x = positions holding X or Y, z = positions holding Y or Z (qubit j <-> bit j%64 of word j//64).
    |c| < tol dropped (BASELINE.json), identity kept (H2 K = 15 counts it).
    """
    lib = _load()
    N = h.shape[0]
    h = np.ascontiguousarray(h, dtype=np.float64)
    g = np.ascontiguousarray(g, dtype=np.float64)
    n = 2 * N
    # upper bound on distinct strings for dense integrals: K(N)
    from math import comb
    kmax = 1 + n + comb(n, 2) + 4 * (n - 1) * comb(N, 2) + 4 * comb(N, 2) ** 2 + 12 * comb(N, 4) + 64
    cap = max(12, int(np.ceil(np.log2(kmax * 2.2))))
    while True:
        x = np.zeros((kmax, 2), dtype=np.uint64)
        z = np.zeros((kmax, 2), dtype=np.uint64)
        c = np.zeros(kmax, dtype=np.float64)
        mi = ctypes.c_double(0.0)
        k = lib.jw_build(N, h.ctypes.data, g.ctypes.data, float(tol), cap, kmax,
                         x.ctypes.data, z.ctypes.data, c.ctypes.data, ctypes.byref(mi))
        if k == -1 and cap < 30:
            cap += 1
            kmax *= 2
            continue
        if k < 0:
            raise RuntimeError(f"jw_build failed ({k})")
        break
    if mi.value > 1e-9:
        raise RuntimeError(f"JW produced non-real coefficients (max |imag| {mi.value:g}): integrals not symmetric?")
    return x[:k].copy(), z[:k].copy(), c[:k].copy()


def masks_to_codes(x: np.ndarray, z: np.ndarray, n_qubits: int) -> np.ndarray:
    """(x, z) masks -> Operator Matrix uint8[K, n] with codes 0..3 = I, X, Y, Z (Eq. 1, Fig. 1)."""
    K = x.shape[0]
    codes = np.zeros((K, n_qubits), dtype=np.uint8)
    for j in range(n_qubits):
        xb = ((x[:, j // 64] >> np.uint64(j % 64)) & np.uint64(1)).astype(np.uint8)
        zb = ((z[:, j // 64] >> np.uint64(j % 64)) & np.uint64(1)).astype(np.uint8)
        # X: x=1,z=0 -> 1 ; Y: x=1,z=1 -> 2 ; Z: x=0,z=1 -> 3
        codes[:, j] = np.where(xb == 1, np.where(zb == 1, 2, 1), np.where(zb == 1, 3, 0))
    return codes


def codes_to_strings(codes: np.ndarray):
    """Operator Matrix -> list of 'IXYZ...' strings (qubit 0 first)."""
    lut = np.array(list("IXYZ"))
    return ["".join(lut[row]) for row in codes]
