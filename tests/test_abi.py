"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/nh.h declares,
validates its arguments, and refuses to compute without a CUDA device (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

import paper_2503_06610_b200 as nh
from paper_2503_06610_b200 import build as nh_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    nh_build.build()
    return nh.load()


def declared_symbols():
    names = set()
    for header in sorted(os.listdir(os.path.join(ROOT, "include"))):      # nh.h (the contract), nh_debug.h (hooks), nh_noalloc.h
        text = open(os.path.join(ROOT, "include", header)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(nh_[a-z_]+)\s*\(", text))
    return sorted(names)


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert set(names) == set(nh.binding.EXPORTS)
    for name in names:
        assert hasattr(lib, name), name


def test_workspace_bytes_and_validation(lib):
    p = nh.make_params(16, 16, 8, 0.8, precision=nh.FP32_SHIFTED)
    N = 16 * 16 * 8
    b32 = nh.workspace_bytes(p)
    # populations A, B; n, n', n^P, a, u, F; FP64 staging; the two-step kernel's plane ring
    # (min(nz-2, 12) planes of 19 populations) and its flags (include/nh.h)
    ring = min(8 - 2, 12) * 19 * 16 * (16 + 2)          # ring planes have two halo rows
    fields32 = (2 * 19 + 6 * 3) * N * 4 + 3 * N * 8 + ring * 4
    assert b32 >= fields32
    assert b32 <= fields32 + 12 * 256 + 8 * (8 + 32 + 2 * 6 * (16 * 18 // 128 + 16 + 3) + 6 + 8)
    p64 = nh.make_params(16, 16, 8, 0.8, precision=nh.FP64_SHIFTED)
    assert nh.workspace_bytes(p64) >= (2 * 19 + 6 * 3) * N * 8 + 3 * N * 8 + ring * 8
    for bad in (dict(tau=0.5), dict(nz=2), dict(gamma1=0.0), dict(K=-1.0), dict(fd_ratio=-1),
                dict(W0=float("inf")), dict(precision=7), dict(anchoring=2), dict(nx=0), dict(coupling=4),
                dict(nx=4096, ny=4096, nz=64)):
        kw = dict(nx=4, ny=4, nz=5, tau=0.8)
        kw.update(bad)
        q = nh.make_params(**kw)
        assert nh.workspace_bytes(q) == 0
        h = C.c_void_p()
        rc = lib.nh_init_lattice(C.byref(q), 256, 1 << 20, None, C.byref(h))
        assert rc == -1 and not h.value
        assert lib.nh_last_error()
    assert nh.workspace_bytes(nh.make_params(512, 512, 128, 0.8)) < 8 * 2 ** 30  # BASELINE: "roughly 7 GB"


def test_slab_calls_reject_null_handles(lib):
    lib.nh_rows_bytes.restype = C.c_size_t
    assert lib.nh_rows_bytes(None, 0, 4) == 0
    assert lib.nh_get_rows(None, 0, 0, 1, 256) == -1 and lib.nh_last_error()
    assert lib.nh_set_rows(None, 0, 0, 1, 256) == -1
    assert lib.nh_update_force(None) == -1
    assert lib.nh_defer_force(None, 1) == -1
    assert lib.nh_get_rows_pair(None, 0, 0, 4, 1, 256) == -1 and b"null handle" in lib.nh_last_error()
    assert lib.nh_set_rows_pair(None, 0, 0, 4, 1, 256) == -1
    assert lib.nh_debug_tune(None, 0, 0) == -1


def test_null_and_small_workspace(lib):
    p = nh.make_params(4, 4, 5, 0.8)
    h = C.c_void_p()
    assert lib.nh_init_lattice(C.byref(p), None, 1 << 20, None, C.byref(h)) == -1
    assert lib.nh_init_lattice(C.byref(p), 256, 16, None, C.byref(h)) == -2
    assert lib.nh_init_lattice(C.byref(p), 257, 1 << 20, None, C.byref(h)) == -1
    assert lib.nh_step(None, 1, 1) == -1
    assert lib.nh_set_director(None, None) == -1
    assert lib.nh_get_fields(None, None, None, None, None) == -1
    assert lib.nh_time(None) == -1
    lib.nh_free(None)


def test_no_cpu_fallback(lib):
    """Without a CUDA device the library must fail loudly, not compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    p = nh.make_params(4, 4, 5, 0.8)
    h = C.c_void_p()
    rc = lib.nh_init_lattice(C.byref(p), 256, 1 << 20, None, C.byref(h))
    assert rc == -3 and not h.value
    assert b"no CUDA device" in lib.nh_last_error()
    with pytest.raises(RuntimeError):
        nh.Lattice(4, 4, 5, 0.8)


def test_product_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package or include/ may reference it."""
    pkg = os.path.join(ROOT, "paper_2503_06610_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src, fn
                assert "nh_oracle" not in src, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_2503_06610_b200 import" not in src and "import paper_2503_06610_b200" not in src, fn
            assert "nh_lb.cuh" not in src and "include/nh.h" not in src, fn


def test_no_alloc_entry_validates_before_it_touches_cuda(lib):
    """nh_lb_two_steps_noalloc (include/nh_noalloc.h): bad arguments and lattices beyond the 16 MiB static scratch are
    refused with NH_EINVAL before any CUDA call; with good arguments and no device it is NH_ECUDA (no CPU path)."""
    g = (C.c_double * 3)(0.0, 0.0, 0.0)
    call = lambda nx, ny, nz, prec, tau, a=4096, b=1 << 40: lib.nh_lb_two_steps_noalloc(nx, ny, nz, prec, tau, g, a, None, b, None)
    assert call(512, 512, 64, 1, 0.8) == -1 and b"beyond the static scratch" in lib.nh_last_error()
    assert call(256, 256, 16, 0, 0.8) == -1 and b"16777216" in lib.nh_last_error()
    assert call(96, 8, 6, 1, 0.8) == -1 and b"nx must be" in lib.nh_last_error()
    assert call(64, 8, 4, 1, 0.8) == -1
    assert call(64, 8, 6, 1, 0.5) == -1
    assert call(64, 8, 6, 9, 0.8) == -1
    assert call(64, 8, 6, 1, 0.8, a=4096, b=4096) == -1 and b"overlap" in lib.nh_last_error()
    assert lib.nh_lb_two_steps_noalloc(64, 8, 6, 1, 0.8, None, 4096, None, 1 << 40, None) == -1
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if not has_gpu:
        assert call(64, 8, 6, 1, 0.8) == -3 and lib.nh_last_error()


def test_binding_constants_equal_the_headers():
    """Every #define of the headers that the binding mirrors has the same value there: options, precisions, fields,
    tuning keys, error codes, the no-alloc scratch size."""
    defs = {}
    for header in ("nh.h", "nh_debug.h", "nh_noalloc.h"):
        text = open(os.path.join(ROOT, "include", header)).read()
        for name, value in re.findall(r"^#define\s+(NH_[A-Z0-9_]+)\s+(\(?[-0-9ux* ]+\)?)", text, flags=re.M):
            defs[name] = eval(value.replace("u", ""))          # plain integer expressions: 16u * 1024u * 1024u
    b = nh.binding
    for name in ("GRAPH", "TIMING", "FD_DIRECT", "NO_SERPENTINE", "FD_NOVEC", "LB_TWOSTEP", "LB_ONESTEP", "CHECK_FINITE"):
        assert getattr(b, "OPT_" + name) == defs["NH_OPT_" + name], name
    for name in ("FP64_SHIFTED", "FP32_SHIFTED", "FP32_UNSHIFTED", "FP64_UNSHIFTED"):
        assert getattr(b, name) == defs["NH_" + name], name
    for i, field in enumerate(b.FIELDS):
        assert defs["NH_FIELD_" + field.upper()] == i
    for key, value in b.TUNE.items():
        assert defs["NH_TUNE_" + key.upper()] == value, key
    assert len(b.TUNE) == defs["NH_TUNE_COUNT"]
    assert b.NOALLOC_SCRATCH_BYTES == defs["NH_NOALLOC_SCRATCH_BYTES"] == 16 * 1024 * 1024
    assert (defs["NH_OK"], defs["NH_EINVAL"], defs["NH_ENOMEM"], defs["NH_ECUDA"], defs["NH_ENUMERIC"]) == (0, -1, -2, -3, -4)
    # option bits are distinct single bits
    bits = [v for k, v in defs.items() if k.startswith("NH_OPT_")]
    assert len(set(bits)) == len(bits) and all(v & (v - 1) == 0 for v in bits)
