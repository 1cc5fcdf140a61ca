"""CPU-side checks of the boundary: libgfmc.so builds for sm_100a, loads, exports every symbol that
include/gfmc.h declares, sizes its workspace on the host, and fails loudly without a GPU / without the
library.  No compute call is made here."""
import ctypes
import re
from pathlib import Path

import pytest

import paper_1303_6016_b200 as g
from paper_1303_6016_b200 import binding
from paper_1303_6016_b200.build import build_library

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    build_library()
    return ctypes.CDLL(str(g.LIB_PATH))


def _declared():
    text = (ROOT / "include" / "gfmc.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gfmc_[a-z_A-Z0-9]+)\s*\(", text)))


def test_header_and_library_agree(lib):
    names = _declared()
    assert {"gfmc_create", "gfmc_set_spins", "gfmc_moments", "gfmc_local_green", "gfmc_sweep", "gfmc_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in gfmc.h but not exported"
    assert sorted(g.EXPORTS) == names


def test_only_gfmc_symbols_are_exported_with_c_linkage(lib):
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", str(g.LIB_PATH)], capture_output=True, text=True).stdout
    syms = [l.split()[-1] for l in out.splitlines() if " T " in l]
    c_syms = [s for s in syms if not s.startswith("_Z") and s not in ("_init", "_fini")]
    assert sorted(c_syms) == _declared()


def test_workspace_bytes_host_only():
    base = dict(L=32, M=1024, n_energy=0, t=1.0, JH=8.0, T=0.02, mu=0.0, kernel=0, lambda_=0.0,
                max_batch_sites=2048, device=0)
    n = g.gfmc_workspace_bytes(**base)
    work_vectors = 2 * 16 * (2 * 32 ** 3) * (2 * 2048)          # two buffers of 16*D*2B bytes
    assert work_vectors <= n <= work_vectors + (1 << 30)
    small = g.gfmc_workspace_bytes(**{**base, "max_batch_sites": 64})
    assert small < n
    for bad in (dict(L=1), dict(M=7), dict(M=0), dict(T=0.0), dict(kernel=5), dict(max_batch_sites=0), dict(L=1000)):
        assert g.gfmc_workspace_bytes(**{**base, **bad}) == 0


def test_params_struct_matches_header():
    text = (ROOT / "include" / "gfmc.h").read_text()
    body = re.search(r"typedef struct gfmc_params \{(.*?)\} gfmc_params;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = [re.sub(r"\s+", " ", f).strip() for f in body.split(";") if f.strip()]
    c_names = [f.split()[-1].lstrip("*") for f in fields]
    py_names = [n.rstrip("_") for n, _ in binding.gfmc_params._fields_]
    assert c_names == py_names


def test_create_without_gpu_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    p = binding.gfmc_params(L=4, M=8, n_energy=0, t=1.0, JH=4.0, T=0.1, mu=0.0, kernel=0, lambda_=4.0,
                            max_batch_sites=1, device=0, stream=None, workspace=None, workspace_bytes=0)
    h = ctypes.c_void_p()
    lib.gfmc_create.argtypes = [ctypes.POINTER(binding.gfmc_params), ctypes.POINTER(ctypes.c_void_p)]
    rc = lib.gfmc_create(ctypes.byref(p), ctypes.byref(h))
    assert rc == -3 and not h.value                     # GFMC_ECUDA, no context
    lib.gfmc_create_error.restype = ctypes.c_char_p
    assert b"no CPU fallback" in lib.gfmc_create_error()
    with pytest.raises(g.GfmcError):
        g.gfmc_create(L=4, M=8, t=1.0, JH=4.0, T=0.1)


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", tmp_path / "libgfmc.so")
    with pytest.raises(FileNotFoundError, match="no fallback"):
        binding.load_library()


def test_product_does_not_import_the_oracle():
    """The product path may not import, link or execute anything under oracle/ (and vice versa)."""
    pat = re.compile(r"^\s*(from|import)\s+oracle|#include.*oracle|gfmc_oracle|libgfmc_oracle", re.M)
    for f in (ROOT / "paper_1303_6016_b200").rglob("*"):
        if f.suffix in (".py", ".cu", ".cuh", ".h"):
            assert not pat.search(f.read_text()), f
    pat2 = re.compile(r"paper_1303_6016_b200|libgfmc\.so|cheb_step|post\.cuh")
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c", ".h"):
            assert not pat2.search(f.read_text().replace("imports nothing from paper_1303_6016_b200", "").replace(
                "(paper_1303_6016_b200/csrc)", "")), f
