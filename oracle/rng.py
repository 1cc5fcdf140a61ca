"""Counter-based random numbers of the Monte Carlo driver (Algorithm 1) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu legs may import this module;
it imports nothing from paper_1303_6016_b200 and shares no code with the CUDA path (which has its own generator kernel).

Algorithm 1 draws two things per trial: "change the spin ... randomly" (line 4) and `rand()` in the acceptance
test (line 10).  The paper does not say which generator; reading f3-1 fixes a COUNTER-BASED one so
that the oracle and the GPU draw identical numbers under any schedule:

    Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11), written out below in plain numpy
    key     = (seed mod 2^32, seed div 2^32)
    counter = (site, sweep mod 2^32, stream, sweep div 2^32)        stream 0 -> (u1, u2), stream 1 -> (u3, unused)
    a 64-bit uniform in [0,1):  u = floor((w_even * 2^32 + w_odd) / 2^11) * 2^-53
    proposal (DESIGN.md §3 recipe, uniform on the sphere):  z = 2 u1 - 1,  phi = 2 pi u2,  S' = (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z)
    acceptance uniform:  u = 1 - u3  in (0, 1]

Pins (tests/test_oracle_rng.py): the three known-answer vectors of the generator's authors (tests/golden/philox4x32_10_kat.txt);
unit norm, range and first/second moments of the derived numbers.
"""
from __future__ import annotations

import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = 0x9E3779B9
_W1 = 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def philox4x32_10(counter, key):
    """counter: four arrays (or ints) of 32-bit words, key: two 32-bit words.  Returns four uint64 arrays holding 32-bit words.
    One round: (c0, c1, c2, c3) <- (hi(M1*c2) ^ c1 ^ k0, lo(M1*c2), hi(M0*c0) ^ c3 ^ k1, lo(M0*c0)); the key is bumped by
    (W0, W1) before every round but the first; ten rounds."""
    c0, c1, c2, c3 = (np.atleast_1d(np.asarray(c, dtype=np.uint64)) & _MASK for c in counter)
    k0, k1 = int(key[0]) & 0xFFFFFFFF, int(key[1]) & 0xFFFFFFFF
    for r in range(10):
        if r > 0:
            k0 = (k0 + _W0) & 0xFFFFFFFF
            k1 = (k1 + _W1) & 0xFFFFFFFF
        p0 = _M0 * c0                      # 32 x 32 -> 64 bit products, exact in uint64
        p1 = _M1 * c2
        n0 = (p1 >> _S32) ^ c1 ^ np.uint64(k0)
        n1 = p1 & _MASK
        n2 = (p0 >> _S32) ^ c3 ^ np.uint64(k1)
        n3 = p0 & _MASK
        c0, c1, c2, c3 = n0, n1, n2, n3
    return c0, c1, c2, c3


def _u01(w_even, w_odd):
    return (((w_even << _S32) | w_odd) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def uniforms(seed: int, sweep: int, N: int):
    """(u1, u2, u3), each [N] in [0,1), for the trial at every site of sweep `sweep`."""
    key = (seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
    site = np.arange(N, dtype=np.uint64)
    lo, hi = sweep & 0xFFFFFFFF, (sweep >> 32) & 0xFFFFFFFF
    a = philox4x32_10((site, np.full(N, lo), np.zeros(N), np.full(N, hi)), key)
    b = philox4x32_10((site, np.full(N, lo), np.ones(N), np.full(N, hi)), key)
    return _u01(a[0], a[1]), _u01(a[2], a[3]), _u01(b[0], b[1])


def proposals(seed: int, sweep: int, N: int):
    """(S'[N,3], u[N]): trial spins uniform on the unit sphere and acceptance uniforms in (0,1], indexed by site."""
    u1, u2, u3 = uniforms(seed, sweep, N)
    z = 2.0 * u1 - 1.0
    r = np.sqrt(1.0 - z * z)
    phi = 2.0 * np.pi * u2
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1), 1.0 - u3


def run_chain(sweep_fn, S, seed: int, first_sweep: int, n_sweeps: int):
    """Algorithm 1 with the generator above.  sweep_fn(S, proposals[1,N,3], uniforms[1,N]) is ONE sweep of the oracle
    (oracle.sweep / oracle.dex_sweep with everything but the spins and the random inputs bound) and returns their dict.
    Returns dict(spins, magnetization[n_sweeps], n_accepted[n_sweeps], dS[n_sweeps,N], accept[n_sweeps,N], proposals, uniforms)."""
    N = S.shape[0]
    out = dict(magnetization=[], n_accepted=[], dS=[], accept=[], proposals=[], uniforms=[])
    for s in range(first_sweep, first_sweep + n_sweeps):
        p, u = proposals(seed, s, N)
        r = sweep_fn(S, p[None], u[None])
        S = r["spins"]
        out["magnetization"].append(r["magnetization"][0]); out["n_accepted"].append(r["n_accepted"][0])
        out["dS"].append(r["dS"][0]); out["accept"].append(r["accept"][0]); out["proposals"].append(p); out["uniforms"].append(u)
    out = {k: np.array(v) for k, v in out.items()}
    out["spins"] = S
    return out
