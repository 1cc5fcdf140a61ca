"""Thin ctypes binding of libgfmc.so (include/gfmc.h).  Argument marshalling only: every step of the
hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory (the workspace
tensor, device-resident inputs/outputs) and for the stream; nothing is computed in Python.

The functions carry the C names (gfmc_create, gfmc_set_spins, gfmc_moments, gfmc_local_green,
gfmc_delta_S, gfmc_update_batch, gfmc_sweep, gfmc_magnetization, gfmc_destroy, ...).  Array arguments may be
numpy arrays (host pointers, mem = GFMC_HOST) or torch CUDA tensors (device pointers, mem = GFMC_DEVICE);
outputs follow the inputs.  There is no CPU fallback: if libgfmc.so is missing or no CUDA device is
present the calls raise.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

GFMC_HOST, GFMC_DEVICE = 0, 1
GFMC_KERNEL_JACKSON, GFMC_KERNEL_LORENTZ, GFMC_KERNEL_NONE = 0, 1, 2
GFMC_MODEL_HUND, GFMC_MODEL_DEX_INF = 0, 1
GFMC_FLAG_NO_RESIDENT, GFMC_FLAG_GREEN_DIRECT, GFMC_FLAG_NO_GRAPH, GFMC_FLAG_TWO_STEP, GFMC_FLAG_NO_PDL = 1, 2, 4, 8, 16
GFMC_BATCH_FROZEN, GFMC_BATCH_EXACT = 0, 1
_ERR = {0: "GFMC_OK", -1: "GFMC_EINVAL", -2: "GFMC_ENOMEM", -3: "GFMC_ECUDA", -4: "GFMC_ESTATE"}

LIB_PATH = Path(__file__).resolve().parent / "libgfmc.so"
_lib = None


class GfmcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_ERR.get(code, code)}: {msg}")
        self.code = code


class gfmc_params(ctypes.Structure):
    _fields_ = [("L", ctypes.c_int32), ("M", ctypes.c_int32), ("n_energy", ctypes.c_int32),
                ("t", ctypes.c_double), ("JH", ctypes.c_double), ("T", ctypes.c_double), ("mu", ctypes.c_double),
                ("kernel", ctypes.c_int32), ("lambda_", ctypes.c_double),
                ("max_batch_sites", ctypes.c_int32), ("device", ctypes.c_int32),
                ("stream", ctypes.c_void_p), ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t),
                ("model", ctypes.c_int32), ("ph_symmetry", ctypes.c_int32),
                ("flags", ctypes.c_int32), ("ring_stages_cur", ctypes.c_int32), ("ring_stages_prev", ctypes.c_int32),
                ("streamk_eff", ctypes.c_double), ("exact_batch_sites", ctypes.c_int32)]


def load_library():
    """dlopen libgfmc.so (built in-tree by __graft_entry__.build()).  Fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise FileNotFoundError(f"{LIB_PATH} not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                                    "(the CUDA path has no fallback)")
        lib = ctypes.CDLL(str(LIB_PATH))
        vp, i32, i64p = ctypes.c_void_p, ctypes.c_int32, ctypes.POINTER(ctypes.c_int64)
        lib.gfmc_workspace_bytes.restype = ctypes.c_size_t
        lib.gfmc_workspace_bytes.argtypes = [ctypes.POINTER(gfmc_params)]
        lib.gfmc_create.argtypes = [ctypes.POINTER(gfmc_params), ctypes.POINTER(vp)]
        lib.gfmc_create_error.restype = ctypes.c_char_p
        lib.gfmc_destroy.argtypes = [vp]
        lib.gfmc_set_spins.argtypes = [vp, vp, ctypes.c_int]
        lib.gfmc_get_spins.argtypes = [vp, vp, ctypes.c_int]
        lib.gfmc_bounds.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        lib.gfmc_moments.argtypes = [vp, vp, i32, vp, ctypes.c_int]
        lib.gfmc_local_green.argtypes = [vp, vp, i32, vp, vp, ctypes.c_int]
        lib.gfmc_delta_S.argtypes = [vp, vp, i32, vp, vp, ctypes.c_int]
        lib.gfmc_update_batch.argtypes = [vp, vp, i32, vp, vp, vp, vp, ctypes.c_int]
        lib.gfmc_decide_batch.argtypes = [vp, vp, i32, vp, vp, vp, vp, ctypes.c_int]
        lib.gfmc_apply_flips.argtypes = [vp, vp, i32, vp, vp, ctypes.c_int]
        lib.gfmc_sweep.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp, ctypes.c_int]
        lib.gfmc_magnetization.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
        lib.gfmc_random_proposals.argtypes = [vp, ctypes.c_uint64, ctypes.c_int64, vp, vp, ctypes.c_int]
        lib.gfmc_run.argtypes = [vp, ctypes.c_uint64, ctypes.c_int64, i32, i32, vp, vp, ctypes.c_int]
        lib.gfmc_set_temperature.argtypes = [vp, ctypes.c_double]
        lib.gfmc_set_batch_mode.argtypes = [vp, ctypes.c_int]
        dp = ctypes.POINTER(ctypes.c_double)
        lib.gfmc_run_summary.argtypes = [vp, dp, dp, dp, i64p]
        lib.gfmc_launch_counts.argtypes = [vp, i64p]
        lib.gfmc_last_step_loop_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_double), i64p]
        lib.gfmc_moments_ov.argtypes = [vp, vp, i32, vp, vp, ctypes.c_int]
        lib.gfmc_local_green_ov.argtypes = [vp, vp, i32, vp, vp, vp, ctypes.c_int]
        lib.gfmc_hopping.argtypes = [vp, vp, ctypes.c_int]
        lib.gfmc_last_step_loop_vectors.argtypes = [vp, i64p, i64p]
        lib.gfmc_last_error.restype = ctypes.c_char_p
        lib.gfmc_last_error.argtypes = [vp]
        lib.gfmc_moments_static.argtypes = [i32, vp, i32, i32, ctypes.c_double, ctypes.c_double, vp, vp, i32, vp]
        lib.gfmc_moments_static_error.restype = ctypes.c_char_p
        lib.gfmc_version.restype = ctypes.c_char_p
        _lib = lib
    return _lib


EXPORTS = ["gfmc_workspace_bytes", "gfmc_create", "gfmc_create_error", "gfmc_destroy", "gfmc_set_spins",
           "gfmc_get_spins", "gfmc_bounds", "gfmc_moments", "gfmc_local_green", "gfmc_delta_S",
           "gfmc_update_batch", "gfmc_decide_batch", "gfmc_apply_flips", "gfmc_sweep", "gfmc_random_proposals", "gfmc_run", "gfmc_run_summary", "gfmc_set_temperature", "gfmc_set_batch_mode", "gfmc_magnetization", "gfmc_launch_counts",
           "gfmc_last_step_loop_ms", "gfmc_last_step_loop_vectors", "gfmc_moments_ov", "gfmc_local_green_ov",
           "gfmc_hopping", "gfmc_last_error", "gfmc_version", "gfmc_moments_static", "gfmc_moments_static_error"]
GFMC_STATIC_MAX_L, GFMC_STATIC_MAX_STEP_SITES = 12, 65536


def _is_torch(x):
    return x is not None and type(x).__module__.startswith("torch")


def _ptr(x):
    if x is None:
        return None
    if _is_torch(x):
        return ctypes.c_void_p(x.data_ptr())
    return ctypes.c_void_p(x.ctypes.data)


def _mem_of(*arrs):
    kinds = {_is_torch(a) for a in arrs if a is not None}
    if len(kinds) > 1:
        raise TypeError("mix of host (numpy) and device (torch) arrays in one call")
    dev = kinds.pop() if kinds else False
    if dev:
        for a in arrs:
            if a is not None and (not a.is_cuda or not a.is_contiguous()):
                raise TypeError("device arguments must be contiguous CUDA tensors")
    return GFMC_DEVICE if dev else GFMC_HOST


def _host(a, dtype, shape=None):
    a = np.ascontiguousarray(a, dtype=dtype)
    if shape is not None and a.shape != tuple(shape):
        raise ValueError(f"expected shape {tuple(shape)}, got {a.shape}")
    return a


class Context:
    """Owner of one gfmc_ctx*.  Created by gfmc_create()."""

    def __init__(self, handle, params, workspace):
        self.handle = handle
        self.params = params
        self.workspace = workspace          # keeps the torch tensor alive
        self.L, self.M = params.L, params.M
        self.N = params.L ** 3
        self.K = params.n_energy if params.n_energy > 0 else 2 * params.M

    def _check(self, rc):
        if rc != 0:
            raise GfmcError(rc, load_library().gfmc_last_error(self.handle).decode())

    def __del__(self):
        try:
            gfmc_destroy(self)
        except Exception:
            pass


def gfmc_create(L, M, t, JH, T, mu=0.0, n_energy=0, kernel=GFMC_KERNEL_JACKSON, lam=4.0,
                max_batch_sites=1, device=0, stream=None, workspace="torch",
                model=GFMC_MODEL_HUND, ph_symmetry=0, flags=0, ring_stages_cur=0, ring_stages_prev=0, streamk_eff=0.0, exact_batch_sites=0) -> Context:
    """workspace: "torch" (default) allocates the arena as a torch.uint8 CUDA tensor and hands its pointer
    to the library; None lets the library cudaMalloc it.  stream: None -> torch's current stream.
    flags / ring_stages_* / streamk_eff: per-context diagnostic overrides (GFMC_FLAG_*, include/gfmc.h); 0 = automatic."""
    lib = load_library()
    p = gfmc_params(L=L, M=M, n_energy=n_energy, t=t, JH=JH, T=T, mu=mu, kernel=kernel, lambda_=lam,
                    max_batch_sites=max_batch_sites, device=device, stream=None, workspace=None, workspace_bytes=0,
                    model=model, ph_symmetry=ph_symmetry, flags=flags, ring_stages_cur=ring_stages_cur,
                    ring_stages_prev=ring_stages_prev, streamk_eff=streamk_eff, exact_batch_sites=exact_batch_sites)
    ws = None
    if workspace == "torch" or stream is None:
        import torch
        if not torch.cuda.is_available():
            raise GfmcError(-3, "no CUDA device (libgfmc has no CPU fallback)")
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        if workspace == "torch":
            nbytes = lib.gfmc_workspace_bytes(ctypes.byref(p))
            if nbytes == 0:
                raise GfmcError(-1, "invalid parameters")
            ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=f"cuda:{device}")
            base = (ws.data_ptr() + 255) // 256 * 256
            p.workspace, p.workspace_bytes = base, nbytes
    p.stream = stream
    h = ctypes.c_void_p()
    rc = lib.gfmc_create(ctypes.byref(p), ctypes.byref(h))
    if rc != 0:
        raise GfmcError(rc, lib.gfmc_create_error().decode())
    return Context(h, p, ws)


def gfmc_destroy(ctx: Context):
    if ctx.handle:
        load_library().gfmc_destroy(ctx.handle)
        ctx.handle = None
        ctx.workspace = None


def gfmc_workspace_bytes(**kw) -> int:
    p = gfmc_params(**kw)
    return load_library().gfmc_workspace_bytes(ctypes.byref(p))


def gfmc_bounds(ctx):
    a, b = ctypes.c_double(), ctypes.c_double()
    ctx._check(load_library().gfmc_bounds(ctx.handle, ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


def gfmc_set_spins(ctx, S):
    if not _is_torch(S):
        S = _host(S, np.float64, (ctx.N, 3))
    ctx._check(load_library().gfmc_set_spins(ctx.handle, _ptr(S), _mem_of(S)))


def gfmc_get_spins(ctx, out=None):
    if out is None:
        out = np.empty((ctx.N, 3), dtype=np.float64)
    ctx._check(load_library().gfmc_get_spins(ctx.handle, _ptr(out), _mem_of(out)))
    return out


def _sites(ctx, sites):
    if _is_torch(sites):
        import torch
        if sites.dtype != torch.int32:
            raise TypeError("device site lists must be int32")
        return sites
    return _host(sites, np.int32)


def _like(ref, shape, dtype_np):
    if _is_torch(ref):
        import torch
        td = {np.float64: torch.float64, np.complex128: torch.complex128, np.uint8: torch.uint8, np.int64: torch.int64}[dtype_np]
        return torch.empty(shape, dtype=td, device=ref.device)
    return np.empty(shape, dtype=dtype_np)


def gfmc_moments(ctx, sites):
    """mu[n_sites, M, 2, 2] complex128: mu[s, n, alpha, beta] = <o_s alpha|T_n(H~)|o_s beta> (undamped)."""
    sites = _sites(ctx, sites)
    n = int(sites.shape[0])
    mu = _like(sites, (n, ctx.M, 2, 2), np.complex128)
    ctx._check(load_library().gfmc_moments(ctx.handle, _ptr(sites), n, _ptr(mu), _mem_of(sites)))
    return mu


def gfmc_moments_static(L, M, t, JH, spins, sites, out=None, stream=None):
    """gfmc_moments for callers that must not allocate device memory inside the library (their own allocator owns the GPU, or an
    allocation call would disturb a stream capture or a latency-critical loop): no context, no workspace; the library's scratch is a
    fixed 4 MiB array in its image, shared by all calls (so calls must not overlap on the GPU).  2 <= L <= 12 and
    (M/2) * n_sites <= GFMC_STATIC_MAX_STEP_SITES, else GfmcError(GFMC_EINVAL).
    spins [L^3, 3] float64 and sites [n] int32 are contiguous CUDA tensors; `out` is a preallocated complex128 CUDA tensor
    [n, M, 2, 2] (pass it to keep this wrapper from asking torch for memory); `stream` a raw cudaStream_t handle (None: torch's
    current stream on that device).  Returns out.  The first call on a device does the one-time set-up; make it before any stream capture."""
    import torch
    if _mem_of(spins, sites, out) != GFMC_DEVICE:
        raise TypeError("gfmc_moments_static takes device tensors")
    if spins.dtype != torch.float64 or tuple(spins.shape) != (L ** 3, 3) or sites.dtype != torch.int32 or sites.dim() != 1:
        raise TypeError("spins must be float64 [L^3, 3] and sites int32 [n]")
    n = int(sites.shape[0])
    if out is None:
        out = torch.empty((n, M, 2, 2), dtype=torch.complex128, device=sites.device)
    elif out.dtype != torch.complex128 or tuple(out.shape) != (n, M, 2, 2) or out.device != sites.device:
        raise TypeError("out must be complex128 [n, M, 2, 2] on the device of sites")
    if stream is None:
        stream = torch.cuda.current_stream(sites.device).cuda_stream
    lib = load_library()
    rc = lib.gfmc_moments_static(sites.device.index or 0, ctypes.c_void_p(stream), L, M, float(t), float(JH),
                                 _ptr(spins), _ptr(sites), n, _ptr(out))
    if rc != 0:
        raise GfmcError(rc, lib.gfmc_moments_static_error().decode())
    return out


def gfmc_local_green(ctx, sites):
    """(E[K] float64 descending, G[n_sites, K, 2, 2] complex128 in physical units)."""
    sites = _sites(ctx, sites)
    n = int(sites.shape[0])
    E = _like(sites, (ctx.K,), np.float64)
    G = _like(sites, (n, ctx.K, 2, 2), np.complex128)
    ctx._check(load_library().gfmc_local_green(ctx.handle, _ptr(sites), n, _ptr(E), _ptr(G), _mem_of(sites)))
    return E, G


def gfmc_moments_ov(ctx, sites, proposals):
    """GFMC_MODEL_DEX_INF: mu[n_sites, M, 2, 2] in the pair (o, v) of Eq. (21) for the trial spins proposals[n_sites, 3]."""
    sites = _sites(ctx, sites)
    n = int(sites.shape[0])
    if not _is_torch(proposals):
        proposals = _host(proposals, np.float64, (n, 3))
    mu = _like(sites, (n, ctx.M, 2, 2), np.complex128)
    ctx._check(load_library().gfmc_moments_ov(ctx.handle, _ptr(sites), n, _ptr(proposals), _ptr(mu), _mem_of(sites, proposals)))
    return mu


def gfmc_local_green_ov(ctx, sites, proposals):
    """GFMC_MODEL_DEX_INF: (E[K], G[n_sites, K, 2, 2] in (o, v), physical units)."""
    sites = _sites(ctx, sites)
    n = int(sites.shape[0])
    if not _is_torch(proposals):
        proposals = _host(proposals, np.float64, (n, 3))
    E = _like(sites, (ctx.K,), np.float64)
    G = _like(sites, (n, ctx.K, 2, 2), np.complex128)
    ctx._check(load_library().gfmc_local_green_ov(ctx.handle, _ptr(sites), n, _ptr(proposals), _ptr(E), _ptr(G),
                                                  _mem_of(sites, proposals)))
    return E, G


def gfmc_hopping(ctx, out=None):
    """GFMC_MODEL_DEX_INF: forward bond amplitudes T[3, N] complex128 of Eq. (3), T[d, i] = t_{i, i+e_d}."""
    if out is None:
        out = np.empty((3, ctx.N), dtype=np.complex128)
    ctx._check(load_library().gfmc_hopping(ctx.handle, _ptr(out), _mem_of(out)))
    return out


def gfmc_delta_S(ctx, sites, proposals):
    sites = _sites(ctx, sites)
    n = int(sites.shape[0])
    if not _is_torch(proposals):
        proposals = _host(proposals, np.float64, (n, 3))
    dS = _like(sites, (n,), np.float64)
    ctx._check(load_library().gfmc_delta_S(ctx.handle, _ptr(sites), n, _ptr(proposals), _ptr(dS), _mem_of(sites, proposals)))
    return dS


def gfmc_update_batch(ctx, sites, proposals, uniforms):
    """One frozen-batch Metropolis update.  Returns (dS[n], accepted[n] uint8)."""
    sites = _sites(ctx, sites)
    n = int(sites.shape[0])
    if not _is_torch(proposals):
        proposals = _host(proposals, np.float64, (n, 3))
        uniforms = _host(uniforms, np.float64, (n,))
    dS = _like(sites, (n,), np.float64)
    acc = _like(sites, (n,), np.uint8)
    ctx._check(load_library().gfmc_update_batch(ctx.handle, _ptr(sites), n, _ptr(proposals), _ptr(uniforms),
                                                _ptr(dS), _ptr(acc), _mem_of(sites, proposals, uniforms)))
    return dS, acc


def gfmc_decide_batch(ctx, sites, proposals, uniforms):
    """gfmc_update_batch without touching the configuration: (dS[n], accepted[n] uint8) of this rank's share of a batch."""
    sites = _sites(ctx, sites)
    n = int(sites.shape[0])
    if not _is_torch(proposals):
        proposals = _host(proposals, np.float64, (n, 3))
        uniforms = _host(uniforms, np.float64, (n,))
    dS = _like(sites, (n,), np.float64)
    acc = _like(sites, (n,), np.uint8)
    ctx._check(load_library().gfmc_decide_batch(ctx.handle, _ptr(sites), n, _ptr(proposals), _ptr(uniforms),
                                                _ptr(dS), _ptr(acc), _mem_of(sites, proposals, uniforms)))
    return dS, acc


def gfmc_apply_flips(ctx, sites, proposals, accepted):
    """S[sites[j]] <- proposals[j] wherever accepted[j] != 0 (the whole batch, all ranks' decisions)."""
    sites = _sites(ctx, sites)
    n = int(sites.shape[0])
    if not _is_torch(proposals):
        proposals = _host(proposals, np.float64, (n, 3))
        accepted = _host(accepted, np.uint8, (n,))
    ctx._check(load_library().gfmc_apply_flips(ctx.handle, _ptr(sites), n, _ptr(proposals), _ptr(accepted),
                                               _mem_of(sites, proposals, accepted)))


def gfmc_sweep(ctx, n_sweeps, batch_sites, proposals, uniforms, want_logs=True):
    """Returns dict(dS, accept, magnetization, n_accepted); proposals [n_sweeps, N, 3], uniforms [n_sweeps, N]."""
    if not _is_torch(proposals):
        proposals = _host(proposals, np.float64, (n_sweeps, ctx.N, 3))
        uniforms = _host(uniforms, np.float64, (n_sweeps, ctx.N))
    dS = _like(proposals, (n_sweeps, ctx.N), np.float64) if want_logs else None
    acc = _like(proposals, (n_sweeps, ctx.N), np.uint8) if want_logs else None
    mag = _like(proposals, (n_sweeps,), np.float64)
    nacc = _like(proposals, (n_sweeps,), np.int64)
    ctx._check(load_library().gfmc_sweep(ctx.handle, n_sweeps, batch_sites, _ptr(proposals), _ptr(uniforms),
                                         _ptr(dS), _ptr(acc), _ptr(mag), _ptr(nacc), _mem_of(proposals, uniforms)))
    return dict(dS=dS, accept=acc, magnetization=mag, n_accepted=nacc)


def gfmc_random_proposals(ctx, seed: int, sweep: int, device: bool = False):
    """(proposals[N,3], uniforms[N]) of sweep `sweep` of chain `seed` from the library's counter-based generator."""
    if device:
        import torch
        prop = torch.empty((ctx.N, 3), dtype=torch.float64, device=f"cuda:{ctx.params.device}")
        uni = torch.empty((ctx.N,), dtype=torch.float64, device=prop.device)
    else:
        prop, uni = np.empty((ctx.N, 3), dtype=np.float64), np.empty(ctx.N, dtype=np.float64)
    ctx._check(load_library().gfmc_random_proposals(ctx.handle, int(seed), int(sweep), _ptr(prop), _ptr(uni), _mem_of(prop)))
    return prop, uni


def gfmc_run(ctx, seed: int, first_sweep: int, n_sweeps: int, batch_sites: int):
    """Algorithm 1 on the device: (magnetization[n_sweeps], n_accepted[n_sweeps]) of sweeps first_sweep .. first_sweep+n_sweeps-1."""
    mag = np.empty(n_sweeps, dtype=np.float64)
    nacc = np.empty(n_sweeps, dtype=np.int64)
    ctx._check(load_library().gfmc_run(ctx.handle, int(seed), int(first_sweep), int(n_sweeps), int(batch_sites), _ptr(mag), _ptr(nacc), 0))
    return mag, nacc


def gfmc_run_summary(ctx):
    """Alg. 1 lines 16-17 for the most recent gfmc_run: dict(mean, stderr, acceptance, n_sweeps), computed by the library."""
    m, e, a, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_double(), ctypes.c_int64()
    ctx._check(load_library().gfmc_run_summary(ctx.handle, ctypes.byref(m), ctypes.byref(e), ctypes.byref(a), ctypes.byref(n)))
    return dict(mean=m.value, stderr=e.value, acceptance=a.value, n_sweeps=int(n.value))


def gfmc_set_batch_mode(ctx, mode: int):
    """GFMC_BATCH_FROZEN (default) or GFMC_BATCH_EXACT (needs exact_batch_sites > 0 at gfmc_create)."""
    ctx._check(load_library().gfmc_set_batch_mode(ctx.handle, int(mode)))


def gfmc_set_temperature(ctx, T: float):
    ctx._check(load_library().gfmc_set_temperature(ctx.handle, float(T)))


def gfmc_magnetization(ctx) -> float:
    m = ctypes.c_double()
    ctx._check(load_library().gfmc_magnetization(ctx.handle, ctypes.byref(m)))
    return m.value


def gfmc_launch_counts(ctx):
    c = (ctypes.c_int64 * 2)()
    ctx._check(load_library().gfmc_launch_counts(ctx.handle, c))
    return int(c[0]), int(c[1])


def gfmc_last_step_loop_ms(ctx):
    ms, n = ctypes.c_double(), ctypes.c_int64()
    ctx._check(load_library().gfmc_last_step_loop_ms(ctx.handle, ctypes.byref(ms), ctypes.byref(n)))
    return ms.value, int(n.value)


def gfmc_last_step_loop_vectors(ctx):
    """(start vectors propagated by the last batch, algorithmic bytes of one fused step over them)."""
    n, b = ctypes.c_int64(), ctypes.c_int64()
    ctx._check(load_library().gfmc_last_step_loop_vectors(ctx.handle, ctypes.byref(n), ctypes.byref(b)))
    return int(n.value), int(b.value)


def gfmc_version() -> str:
    return load_library().gfmc_version().decode()
