"""ctypes front end of oracle/me_oracle.c (argument marshalling only; all arithmetic is in the C file).

TEST INFRASTRUCTURE, NOT PRODUCT.  The oracle follows SURVEY.md §8(c): colour-ordered Berends-Giele
recursion + brute-force SU(3) colour matrix for g g -> t tbar + (n-2) g, explicit Dirac algebra for
e+ e- -> mu+ mu-.  Conventions, readings and pins are listed in the C header and in DESIGN.md.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from functools import lru_cache

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "me_oracle.c")

# number of gluons per process and the averaging/symmetry factor denom (reading A3):
# gg initial state 2*2 spins * 8*8 colours = 256, times (n-2)! for identical final gluons; e+e-: 2*2.
NGLUONS = {"gg_ttx": 2, "gg_ttxg": 3, "gg_ttxgg": 4, "gg_ttxggg": 5, "gg_ttxgggg": 6}
DENOM = {"epem_mupmum": 4.0, "gg_ttx": 256.0, "gg_ttxg": 256.0, "gg_ttxgg": 512.0, "gg_ttxggg": 1536.0,
         "gg_ttxgggg": 6144.0}


def _lib_path(long_double: bool) -> str:
    return os.path.join(_HERE, "liboracle_ld.so" if long_double else "liboracle.so")


def build(force: bool = False) -> None:
    """Compile the C oracle (gcc -O2 -fopenmp), both the fp64 and the long-double arbiter build."""
    for ld in (False, True):
        out = _lib_path(ld)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-o", out, _SRC, "-lm"]
        if ld:
            cmd.insert(1, "-DORC_LONG_DOUBLE")
        subprocess.check_call(cmd)


@lru_cache(maxsize=None)
def _lib(long_double: bool = False) -> ctypes.CDLL:
    build()
    lib = ctypes.CDLL(_lib_path(long_double))
    dp = ctypes.POINTER(ctypes.c_double)
    ip = ctypes.POINTER(ctypes.c_int)
    lib.orc_color_matrix.argtypes = [ctypes.c_int, dp, dp]
    lib.orc_color_matrix.restype = ctypes.c_int
    lib.orc_color_matrix_row0.argtypes = [ctypes.c_int, dp, dp]
    lib.orc_color_matrix_row0.restype = ctypes.c_int
    lib.orc_ggttx_partial.argtypes = [ctypes.c_int, dp, ip, ctypes.c_double, ctypes.c_double, ctypes.c_double, dp, dp]
    lib.orc_ggttx_partial.restype = ctypes.c_int
    lib.orc_me_ggttx.argtypes = [ctypes.c_int, dp, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                 dp, ctypes.c_double, dp, dp]
    lib.orc_me_ggttx.restype = ctypes.c_int
    lib.orc_me_eemumu.argtypes = [dp, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                  dp, dp]
    lib.orc_me_eemumu.restype = ctypes.c_int
    lib.orc_su3_generators.argtypes = [dp]
    lib.orc_real_bits.restype = ctypes.c_int
    return lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def su3_generators() -> np.ndarray:
    """T^a = lambda^a/2 as used by the oracle, complex [8][3][3]."""
    out = np.zeros((8, 3, 3, 2))
    _lib().orc_su3_generators(_dp(out))
    return out[..., 0] + 1j * out[..., 1]


def color_matrix_from_row0(n: int):
    """(C, max |imag|) with C_{s s'} = C_{id, s^-1 o s'} filled from the brute-force first row (orc_color_matrix_row0)."""
    import itertools
    nperm = math.factorial(n)
    row = np.zeros(nperm)
    mi = ctypes.c_double(0.0)
    if _lib().orc_color_matrix_row0(n, _dp(row), ctypes.byref(mi)) != nperm:
        raise RuntimeError("orc_color_matrix_row0 failed")
    perms = list(itertools.permutations(range(n)))            # lexicographic, like perms_lex in the C file
    rank = {p: i for i, p in enumerate(perms)}
    C = np.zeros((nperm, nperm))
    for i, s in enumerate(perms):
        inv = [0] * n
        for pos, g in enumerate(s):
            inv[g] = pos
        C[i] = row[[rank[tuple(inv[g] for g in t)] for t in perms]]
    return C, mi.value


@lru_cache(maxsize=None)
def _color_matrix_cached(n: int):
    if n >= 6:
        return color_matrix_from_row0(n)
    nperm = math.factorial(n)
    C = np.zeros((nperm, nperm))
    mi = ctypes.c_double(0.0)
    r = _lib().orc_color_matrix(n, _dp(C), ctypes.byref(mi))
    if r != nperm:
        raise RuntimeError("orc_color_matrix failed")
    return C, mi.value


def color_matrix(n: int) -> np.ndarray:
    """C_{sigma sigma'} for n gluons, brute force over SU(3) indices, permutations in lexicographic order."""
    return _color_matrix_cached(n)[0].copy()


def color_matrix_max_imag(n: int) -> float:
    return _color_matrix_cached(n)[1]


def partial_amplitudes(n: int, mom: np.ndarray, hel, mt: float, wt: float, gs: float,
                       eps_override: np.ndarray | None = None, long_double: bool = False) -> np.ndarray:
    """A(sigma) [n!] complex for one event (mom [n+2][4]) and one helicity assignment (+-1 per particle)."""
    mom = np.ascontiguousarray(mom, dtype=np.float64)
    helc = (ctypes.c_int * (n + 2))(*[int(h) for h in hel])
    A = np.zeros((math.factorial(n), 2))
    eo = None
    if eps_override is not None:
        e = np.asarray(eps_override, dtype=np.complex128)
        eo = np.ascontiguousarray(np.stack([e.real, e.imag], axis=-1))
    r = _lib(long_double).orc_ggttx_partial(n, _dp(mom), helc, mt, wt, gs, _dp(eo) if eo is not None else None, _dp(A))
    if r < 0:
        raise RuntimeError("orc_ggttx_partial failed")
    return A[:, 0] + 1j * A[:, 1]


def me_ggttx(n: int, mom: np.ndarray, mt: float, wt: float, gs: float, denom: float | None = None,
             per_helicity: bool = False, long_double: bool = False):
    mom = np.ascontiguousarray(mom, dtype=np.float64)
    nevt = mom.shape[0]
    assert mom.shape[1:] == (n + 2, 4)
    C = color_matrix(n)
    if denom is None:
        denom = 256.0 * math.factorial(n - 2)
    me = np.zeros(nevt)
    mh = np.zeros((nevt, 1 << (n + 2))) if per_helicity else None
    r = _lib(long_double).orc_me_ggttx(n, _dp(mom), nevt, mt, wt, gs, _dp(C), denom, _dp(me),
                                       _dp(mh) if mh is not None else None)
    if r != 0:
        raise RuntimeError("orc_me_ggttx failed")
    return (me, mh) if per_helicity else me


def me_eemumu(mom: np.ndarray, alpha: float, mZ: float, wZ: float, mW: float, per_helicity: bool = False,
              long_double: bool = False):
    mom = np.ascontiguousarray(mom, dtype=np.float64)
    nevt = mom.shape[0]
    assert mom.shape[1:] == (4, 4)
    me = np.zeros(nevt)
    mh = np.zeros((nevt, 16)) if per_helicity else None
    r = _lib(long_double).orc_me_eemumu(_dp(mom), nevt, alpha, mZ, wZ, mW, _dp(me), _dp(mh) if mh is not None else None)
    if r != 0:
        raise RuntimeError("orc_me_eemumu failed")
    return (me, mh) if per_helicity else me


def matrix_elements(process: str, mom: np.ndarray, params: dict, per_helicity: bool = False, long_double: bool = False):
    """me[nevt] (and me_hel[nevt][ncomb]) for one of the five processes with a parameter card
    {aEWM1, mZ, wZ, mW, mT, wT, aS} (same keys as the C-ABI's mg_set_parameters)."""
    if process == "epem_mupmum":
        return me_eemumu(mom, 1.0 / params["aEWM1"], params["mZ"], params["wZ"], params["mW"], per_helicity, long_double)
    n = NGLUONS[process]
    gs = math.sqrt(4.0 * math.pi * params["aS"])
    return me_ggttx(n, mom, params["mT"], params["wT"], gs, DENOM[process], per_helicity, long_double)
