"""ctypes binding of oracle/gfmc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from paper_1303_6016_b200.
Argument marshalling only: every number is computed by the C file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gfmc_oracle.c"
_SRC_DEX = _HERE / "gfmc_oracle_dex.c"      # J_H -> infinity Hamiltonian, Eq. (2)-(3), (15)-(22)
_SRC_EXACT = _HERE / "gfmc_oracle_exact.c"  # exactness inside a batch: cross moments + Dyson update
_LIB = _HERE / "libgfmc_oracle.so"
_lib = None

c_double_p = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> Path:
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the .so."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < max(p.stat().st_mtime for p in (_SRC, _SRC_DEX, _SRC_EXACT)):
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp",
                               "-ffp-contract=off", str(_SRC), str(_SRC_DEX), str(_SRC_EXACT), "-o", str(tmp), "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(str(_LIB))
        _lib.gfmc_oracle_delta_S.restype = ctypes.c_double
        _lib.gfmc_oracle_magnetization.restype = ctypes.c_double
        _lib.gfmc_oracle_dex_delta_S.restype = ctypes.c_double
    return _lib


def _p(a, ctype=ctypes.c_void_p):
    return a.ctypes.data_as(ctype) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def bounds(t: float, JH: float):
    a, b = ctypes.c_double(), ctypes.c_double()
    lib().gfmc_oracle_bounds(ctypes.c_double(t), ctypes.c_double(JH), ctypes.byref(a), ctypes.byref(b))
    return a.value, b.value


def apply_H(L, t, JH, S, x):
    S, x = _f64(S), _c128(x)
    y = np.empty_like(x)
    lib().gfmc_oracle_apply_H(L, ctypes.c_double(t), ctypes.c_double(JH), _p(S), _p(x), _p(y))
    return y


def moments(L, t, JH, S, site, M):
    """mu[M,2,2] complex: mu[n,alpha,beta] = <o alpha|T_n(H~)|o beta> (undamped)."""
    S = _f64(S)
    mu = np.empty((M, 2, 2), dtype=np.complex128)
    rc = lib().gfmc_oracle_moments(L, ctypes.c_double(t), ctypes.c_double(JH), _p(S), int(site), int(M), _p(mu))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_moments rc={rc}")
    return mu


def moments_many(L, t, JH, S, sites, M, nthreads=1):
    S = _f64(S)
    sites = np.ascontiguousarray(sites, dtype=np.int32)
    mu = np.empty((len(sites), M, 2, 2), dtype=np.complex128)
    rc = lib().gfmc_oracle_moments_many(L, ctypes.c_double(t), ctypes.c_double(JH), _p(S), _p(sites),
                                        len(sites), int(M), _p(mu), int(nthreads))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_moments_many rc={rc}")
    return mu


def kernel(kind, M, lam=4.0):
    g = np.empty(M, dtype=np.float64)
    rc = lib().gfmc_oracle_kernel(int(kind), int(M), ctypes.c_double(lam), _p(g))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_kernel rc={rc}")
    return g


def green(mu, K, kind, lam, a, b):
    """Returns (E[K] physical energies, Gt[K,2,2] = G~; physical G = G~/a)."""
    mu = _c128(mu)
    M = mu.shape[0]
    E = np.empty(K, dtype=np.float64)
    Gt = np.empty((K, 2, 2), dtype=np.complex128)
    rc = lib().gfmc_oracle_green(int(M), int(K), _p(mu), int(kind), ctypes.c_double(lam),
                                 ctypes.c_double(a), ctypes.c_double(b), _p(E), _p(Gt))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_green rc={rc}")
    return E, Gt


def delta_S(Gt, S_old, S_new, JH, a, b, T, mu_chem=0.0, want_theta=False):
    Gt = _c128(Gt)
    K = Gt.shape[0]
    S_old, S_new = _f64(S_old), _f64(S_new)
    theta = np.empty(K, dtype=np.float64) if want_theta else None
    d = np.empty(K, dtype=np.complex128) if want_theta else None
    val = lib().gfmc_oracle_delta_S(int(K), _p(Gt), _p(S_old), _p(S_new), ctypes.c_double(JH),
                                    ctypes.c_double(a), ctypes.c_double(b), ctypes.c_double(T),
                                    ctypes.c_double(mu_chem), _p(theta), _p(d))
    return (val, theta, d) if want_theta else val


def magnetization(S):
    S = _f64(S)
    return lib().gfmc_oracle_magnetization(int(S.shape[0]), _p(S))


def site_dS(L, t, JH, T, mu_chem, M, K, kind, lam, S, site, S_new):
    S, S_new = _f64(S), _f64(S_new)
    out = ctypes.c_double()
    rc = lib().gfmc_oracle_site_dS(L, ctypes.c_double(t), ctypes.c_double(JH), ctypes.c_double(T),
                                   ctypes.c_double(mu_chem), int(M), int(K), int(kind), ctypes.c_double(lam),
                                   _p(S), int(site), _p(S_new), ctypes.byref(out))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_site_dS rc={rc}")
    return out.value


def sweep(L, t, JH, T, mu_chem, M, K, kind, lam, S, n_sweeps, batch_sites, proposals, uniforms, nthreads=1):
    """Runs n_sweeps frozen-batch sweeps.  Returns dict with the updated spins and logs."""
    S = _f64(S).copy()
    N = L ** 3
    proposals, uniforms = _f64(proposals), _f64(uniforms)
    assert proposals.shape == (n_sweeps, N, 3) and uniforms.shape == (n_sweeps, N)
    dS = np.zeros((n_sweeps, N), dtype=np.float64)
    acc = np.zeros((n_sweeps, N), dtype=np.uint8)
    mag = np.zeros(n_sweeps, dtype=np.float64)
    nacc = np.zeros(n_sweeps, dtype=np.int64)
    rc = lib().gfmc_oracle_sweep(L, ctypes.c_double(t), ctypes.c_double(JH), ctypes.c_double(T),
                                 ctypes.c_double(mu_chem), int(M), int(K), int(kind), ctypes.c_double(lam),
                                 _p(S), int(n_sweeps), int(batch_sites), _p(proposals), _p(uniforms),
                                 _p(dS), _p(acc), _p(mag), _p(nacc), int(nthreads))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_sweep rc={rc}")
    return dict(spins=S, dS=dS, accept=acc, magnetization=mag, n_accepted=nacc)


# ----------------------------------------------------------------------------- J_H -> infinity (gfmc_oracle_dex.c)
def dex_bounds(t: float):
    a, b = ctypes.c_double(), ctypes.c_double()
    lib().gfmc_oracle_dex_bounds(ctypes.c_double(t), ctypes.byref(a), ctypes.byref(b))
    return a.value, b.value


def dex_hopping(Si, Sj) -> complex:
    """t_ij of Eq. (3)."""
    Si, Sj = _f64(Si), _f64(Sj)
    out = np.empty(2, dtype=np.float64)
    lib().gfmc_oracle_dex_hopping(_p(Si), _p(Sj), _p(out))
    return complex(out[0], out[1])


def dex_apply_H(L, t, S, x):
    S, x = _f64(S), _c128(x)
    y = np.empty_like(x)
    lib().gfmc_oracle_dex_apply_H(L, ctypes.c_double(t), _p(S), _p(x), _p(y))
    return y


def dex_v(L, t, S, site, S_new):
    """(nb[6] int32, v[6] complex): |v> = Delta|o> = sum_j v_j |nb_j>, Eq. (21)."""
    S, S_new = _f64(S), _f64(S_new)
    nb = np.empty(6, dtype=np.int32)
    v = np.empty(6, dtype=np.complex128)
    lib().gfmc_oracle_dex_v(L, ctypes.c_double(t), _p(S), int(site), _p(S_new), _p(nb), _p(v))
    return nb, v


def dex_moments(L, t, S, site, S_new, M):
    """mu[M,2,2]: <alpha|T_n(H~)|beta>, alpha, beta in (o, v)."""
    S, S_new = _f64(S), _f64(S_new)
    mu = np.empty((M, 2, 2), dtype=np.complex128)
    rc = lib().gfmc_oracle_dex_moments(L, ctypes.c_double(t), _p(S), int(site), _p(S_new), int(M), _p(mu))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_dex_moments rc={rc}")
    return mu


def dex_moments_many(L, t, S, sites, S_new, M, nthreads=1):
    S, S_new = _f64(S), _f64(S_new)
    sites = np.ascontiguousarray(sites, dtype=np.int32)
    assert S_new.shape == (len(sites), 3)
    mu = np.empty((len(sites), M, 2, 2), dtype=np.complex128)
    rc = lib().gfmc_oracle_dex_moments_many(L, ctypes.c_double(t), _p(S), _p(sites), len(sites), _p(S_new),
                                            int(M), _p(mu), int(nthreads))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_dex_moments_many rc={rc}")
    return mu


def dex_delta_S(Gt, a, b, T, mu_chem=0.0, want_theta=False):
    Gt = _c128(Gt)
    K = Gt.shape[0]
    theta = np.empty(K, dtype=np.float64) if want_theta else None
    d = np.empty(K, dtype=np.complex128) if want_theta else None
    val = lib().gfmc_oracle_dex_delta_S(int(K), _p(Gt), ctypes.c_double(a), ctypes.c_double(b), ctypes.c_double(T),
                                        ctypes.c_double(mu_chem), _p(theta), _p(d))
    return (val, theta, d) if want_theta else val


def dex_site_dS(L, t, T, mu_chem, M, K, kind, lam, S, site, S_new):
    S, S_new = _f64(S), _f64(S_new)
    out = ctypes.c_double()
    rc = lib().gfmc_oracle_dex_site_dS(L, ctypes.c_double(t), ctypes.c_double(T), ctypes.c_double(mu_chem), int(M), int(K),
                                       int(kind), ctypes.c_double(lam), _p(S), int(site), _p(S_new), ctypes.byref(out))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_dex_site_dS rc={rc}")
    return out.value


def dex_sweep(L, t, T, mu_chem, M, K, kind, lam, S, n_sweeps, batch_sites, proposals, uniforms, nthreads=1):
    S = _f64(S).copy()
    N = L ** 3
    proposals, uniforms = _f64(proposals), _f64(uniforms)
    assert proposals.shape == (n_sweeps, N, 3) and uniforms.shape == (n_sweeps, N)
    dS = np.zeros((n_sweeps, N), dtype=np.float64)
    acc = np.zeros((n_sweeps, N), dtype=np.uint8)
    mag = np.zeros(n_sweeps, dtype=np.float64)
    nacc = np.zeros(n_sweeps, dtype=np.int64)
    rc = lib().gfmc_oracle_dex_sweep(L, ctypes.c_double(t), ctypes.c_double(T), ctypes.c_double(mu_chem), int(M), int(K),
                                     int(kind), ctypes.c_double(lam), _p(S), int(n_sweeps), int(batch_sites),
                                     _p(proposals), _p(uniforms), _p(dS), _p(acc), _p(mag), _p(nacc), int(nthreads))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_dex_sweep rc={rc}")
    return dict(spins=S, dS=dS, accept=acc, magnetization=mag, n_accepted=nacc)


# ----------------------------------------------------------------------------- exactness inside a batch (gfmc_oracle_exact.c)
def cross_moments(L, t, JH, S, sites, M, nthreads=1):
    """mu[n,n,M,2,2]: mu[X,Y,m,al,be] = <o_X al|T_m(H~)|o_Y be> (direct read-out of the plain recursion)."""
    S = _f64(S)
    sites = np.ascontiguousarray(sites, dtype=np.int32)
    n = len(sites)
    mu = np.empty((n, n, M, 2, 2), dtype=np.complex128)
    rc = lib().gfmc_oracle_cross_moments(L, ctypes.c_double(t), ctypes.c_double(JH), _p(S), _p(sites), n, int(M), _p(mu), int(nthreads))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_cross_moments rc={rc}")
    return mu


def exact_batch(Gt, S_old, S_new, uniforms, JH, a, b, T, mu_chem=0.0, want_d=False):
    """Gt[n,n,K,2,2] = G~ blocks between the sites of a batch at batch start.  Returns (dS[n], accept[n][, d[n,K]])."""
    Gt = _c128(Gt)
    n, K = Gt.shape[0], Gt.shape[2]
    S_old, S_new, uniforms = _f64(S_old), _f64(S_new), _f64(uniforms)
    assert Gt.shape == (n, n, K, 2, 2) and S_old.shape == (n, 3) and S_new.shape == (n, 3) and uniforms.shape == (n,)
    dS = np.empty(n, dtype=np.float64)
    acc = np.empty(n, dtype=np.uint8)
    d = np.empty((n, K), dtype=np.complex128) if want_d else None
    rc = lib().gfmc_oracle_exact_batch(int(K), int(n), _p(Gt), _p(S_old), _p(S_new), _p(uniforms), ctypes.c_double(JH),
                                       ctypes.c_double(a), ctypes.c_double(b), ctypes.c_double(T), ctypes.c_double(mu_chem),
                                       _p(dS), _p(acc), _p(d))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_exact_batch rc={rc}")
    return (dS, acc, d) if want_d else (dS, acc)


def exact_batch_dS(L, t, JH, T, mu_chem, M, K, kind, lam, S, sites, proposals, uniforms, nthreads=1):
    """(dS[n], accept[n]) of the batch `sites` against S, exact inside the batch; proposals[n,3], uniforms[n] by position."""
    S, proposals, uniforms = _f64(S), _f64(proposals), _f64(uniforms)
    sites = np.ascontiguousarray(sites, dtype=np.int32)
    n = len(sites)
    dS = np.empty(n, dtype=np.float64)
    acc = np.empty(n, dtype=np.uint8)
    rc = lib().gfmc_oracle_exact_batch_dS(L, ctypes.c_double(t), ctypes.c_double(JH), ctypes.c_double(T), ctypes.c_double(mu_chem),
                                          int(M), int(K), int(kind), ctypes.c_double(lam), _p(S), _p(sites), n,
                                          _p(proposals), _p(uniforms), _p(dS), _p(acc), int(nthreads))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_exact_batch_dS rc={rc}")
    return dS, acc


def sweep_exact(L, t, JH, T, mu_chem, M, K, kind, lam, S, n_sweeps, batch_sites, proposals, uniforms, nthreads=1):
    """oracle.sweep with the decisions inside every batch taken sequentially and exactly (Dyson update of G)."""
    S = _f64(S).copy()
    N = L ** 3
    proposals, uniforms = _f64(proposals), _f64(uniforms)
    assert proposals.shape == (n_sweeps, N, 3) and uniforms.shape == (n_sweeps, N)
    dS = np.zeros((n_sweeps, N), dtype=np.float64)
    acc = np.zeros((n_sweeps, N), dtype=np.uint8)
    mag = np.zeros(n_sweeps, dtype=np.float64)
    nacc = np.zeros(n_sweeps, dtype=np.int64)
    rc = lib().gfmc_oracle_sweep_exact(L, ctypes.c_double(t), ctypes.c_double(JH), ctypes.c_double(T),
                                       ctypes.c_double(mu_chem), int(M), int(K), int(kind), ctypes.c_double(lam),
                                       _p(S), int(n_sweeps), int(batch_sites), _p(proposals), _p(uniforms),
                                       _p(dS), _p(acc), _p(mag), _p(nacc), int(nthreads))
    if rc != 0:
        raise RuntimeError(f"gfmc_oracle_sweep_exact rc={rc}")
    return dict(spins=S, dS=dS, accept=acc, magnetization=mag, n_accepted=nacc)
