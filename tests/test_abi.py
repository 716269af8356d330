"""CPU-only checks of the boundary: the library builds, loads, exports every symbol the header
declares, validates arguments, and fails loudly (no CPU fallback) when there is no device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1309_1599_b200 import build, binding
    build.build()
    return binding.load_library()


def header_symbols():
    text = open(os.path.join(ROOT, "include", "sg_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sg_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    from paper_1309_1599_b200 import binding
    syms = header_symbols()
    assert sorted(binding.DECLARED_SYMBOLS) == syms
    for s in syms:
        assert hasattr(lib, s), s


def test_host_philox_known_answers(lib):
    from paper_1309_1599_b200 import binding
    rows = [l.split() for l in open(os.path.join(ROOT, "tests", "golden", "philox4x32_10_kat.txt")) if not l.startswith("#")]
    for r in rows:
        v = [int(t, 16) for t in r if t != "->"]
        assert binding.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_workspace_bytes_and_shape_validation(lib):
    from paper_1309_1599_b200 import binding
    wb = binding.workspace_bytes
    assert wb(4, 1, 2, 4) > 0
    # cfg 4: spins 2.42 GB + gathered couplings + raw couplings + staging, well under 180 GB
    b4 = wb(64, 4, 4, 48)
    assert 2.4e9 < b4 < 4e9
    assert wb(5, 1, 2, 4) == 0          # odd L: no periodic checkerboard (reading R4)
    assert wb(0, 1, 2, 4) == 0 and wb(4, 0, 2, 4) == 0 and wb(4, 1, 0, 4) == 0 and wb(4, 1, 2, 0) == 0
    assert wb(4, 1, 2, 4, first_sample=-1) == 0
    assert wb(2, 1, 1, 1) > 0           # smallest legal shape


def test_create_rejects_bad_arguments_without_a_device(lib):
    from paper_1309_1599_b200 import binding
    shape = binding.SgShape(4, 1, 2, 4, 0, 0, 0, 0, 1)
    ctx = ctypes.c_void_p()
    betas = np.array([0.6, 0.9, 1.2, 1.6])
    fake = ctypes.c_void_p(256 * 1000)
    big = 1 << 30
    call = lambda sh, b, ws, n: lib.sg_create(ctypes.byref(ctx), ctypes.byref(sh), b, ws, n, None)
    bp = lambda a: ctypes.c_void_p(a.ctypes.data)
    assert call(shape, None, fake, big) == binding.SG_EINVAL
    assert call(shape, bp(betas), None, big) == binding.SG_EINVAL
    assert call(shape, bp(betas), ctypes.c_void_p(256 * 1000 + 4), big) == binding.SG_EINVAL      # misaligned
    assert call(shape, bp(betas), fake, 16) == binding.SG_EINVAL                                   # too small
    assert call(shape, bp(np.array([0.6, 0.9, 0.9, 1.6])), fake, big) == binding.SG_EINVAL         # not strictly monotone
    assert call(shape, bp(np.array([0.6, np.nan, 1.2, 1.6])), fake, big) == binding.SG_EINVAL
    assert call(shape, bp(np.array([0.6, 1.2, 0.9, 1.6])), fake, big) == binding.SG_EINVAL
    assert call(binding.SgShape(3, 1, 2, 4, 0, 0, 0, 0, 1), bp(betas), fake, big) == binding.SG_EINVAL
    # replica sharding: the window [first_replica, first_replica + n_replicas) must lie inside n_replicas_total
    assert call(binding.SgShape(4, 1, 2, 4, 0, 3, 4, 0, 1), bp(betas), fake, big) == binding.SG_EINVAL
    assert call(binding.SgShape(4, 1, 2, 4, 0, 1, 0, 0, 1), bp(betas), fake, big) == binding.SG_EINVAL
    assert call(binding.SgShape(4, 1, 2, 4, 0, -1, 4, 0, 1), bp(betas), fake, big) == binding.SG_EINVAL
    assert call(binding.SgShape(4, 1, 2, 4, 0, 0, 0, 7, 1), bp(betas), fake, big) == binding.SG_EINVAL   # unknown flag bits
    assert call(binding.SgShape(4, 1, 2, 4, 0, 0, 0, 1, 1), bp(betas), fake, big) == binding.SG_EINVAL   # fused buffer: L % 8 != 0
    # temperature-slot sharding: n_temps_total a multiple of n_temps, first_slot a multiple of n_temps inside it
    assert call(binding.SgShape(4, 1, 2, 4, 0, 0, 0, 0, 1, 0, 6), bp(betas), fake, big) == binding.SG_EINVAL
    assert call(binding.SgShape(4, 1, 2, 4, 0, 0, 0, 0, 1, 2, 8), bp(betas), fake, big) == binding.SG_EINVAL
    assert call(binding.SgShape(4, 1, 2, 4, 0, 0, 0, 0, 1, 8, 8), bp(betas), fake, big) == binding.SG_EINVAL
    assert call(binding.SgShape(4, 1, 2, 4, 0, 0, 0, 0, 1, 4, 0), bp(betas), fake, big) == binding.SG_EINVAL
    assert ctx.value is None
    for fn in (lib.sg_pt_publish, lib.sg_pt_swap_gathered):
        assert fn(None, None) == binding.SG_EINVAL
    assert lib.sg_energy_by_temp(None, None, None) == binding.SG_EINVAL and lib.sg_pt_visits(None, None) == binding.SG_EINVAL
    assert np.isnan(lib.sg_walk_tau_int(None, 10, 0.0))
    for fn in (lib.sg_sweep_or, lib.sg_sweep_hb):
        assert fn(None, 1) == binding.SG_EINVAL
    assert lib.sg_pt_swap(None) == binding.SG_EINVAL
    assert lib.sg_measure(None, None, None, None) == binding.SG_EINVAL
    assert lib.sg_strerror(binding.SG_ECUDA).decode().startswith("CUDA")
    # the widened entry points reject a NULL context too (no device needed)
    assert lib.sg_accumulate(None, 0) == binding.SG_EINVAL and lib.sg_get_logbins(None, None, None, None) == binding.SG_EINVAL
    assert lib.sg_pt_walk(None, None, None) == binding.SG_EINVAL
    assert lib.sg_init_sample_bimodal(None, 0, 0.5, None, None) == binding.SG_EINVAL
    assert lib.sg_export_replica(None, 0, None) == binding.SG_EINVAL and lib.sg_measure_cross(None, 0, None, None, None) == binding.SG_EINVAL
    assert lib.sg_export_chirality(None, 0, None) == binding.SG_EINVAL and lib.sg_chiral_cross(None, None, None, None, None) == binding.SG_EINVAL
    assert lib.sg_measure_chiral(None, None, None) == binding.SG_EINVAL and lib.sg_schwinger_dyson(None, None) == binding.SG_EINVAL


def test_static_entry_point_validates_before_touching_the_device(lib):
    """sg_chiral_cross_static checks its arguments and its fixed capacity before any CUDA call, so the codes can be
    checked without a device: NULL / bad shapes -> SG_EINVAL, a shape beyond SG_STATIC_SCRATCH_BYTES -> SG_ELIMIT."""
    from paper_1309_1599_b200 import binding
    p = ctypes.c_void_p(4096)      # never dereferenced: every call below is rejected first
    err = ctypes.c_int(7)
    call = lambda L, S, T, a=p, b=p, o=p: lib.sg_chiral_cross_static(L, S, T, a, b, o, None, ctypes.byref(err))
    assert call(8, 1, 4, a=None) == binding.SG_EINVAL and call(8, 1, 4, b=None) == binding.SG_EINVAL
    assert call(8, 1, 4, o=None) == binding.SG_EINVAL and call(8, 1, 4, o=ctypes.c_void_p(4100)) == binding.SG_EINVAL
    assert err.value == 0                                                         # cleared on entry
    for L, S, T in ((7, 1, 4), (0, 1, 4), (binding.STATIC_MAX_L + 2, 1, 4), (8, 0, 4), (8, 1, 0), (8, 1, 257)):
        assert call(L, S, T) == binding.SG_EINVAL, (L, S, T)
    # capacity: 4096 + S * 128 * ((256 // T) * T) * 21 * 8 bytes against the fixed 16 MiB
    need = lambda S, T: 4096 + S * 128 * ((256 // T) * T) * 21 * 8
    for S, T in ((4, 256), (4, 48), (4, 1), (7, 129), (100, 3)):
        assert need(S, T) > binding.STATIC_SCRATCH_BYTES
        assert call(8, S, T) == binding.SG_ELIMIT, (S, T)
    assert need(3, 256) <= binding.STATIC_SCRATCH_BYTES and need(6, 130) <= binding.STATIC_SCRATCH_BYTES < need(6, 131)
    assert call(8, 6, 131) == binding.SG_ELIMIT
    msg = lib.sg_strerror(binding.SG_ELIMIT).decode()
    assert "SG_STATIC_SCRATCH_BYTES" in msg and "split" in msg
    text = open(os.path.join(ROOT, "include", "sg_b200.h")).read()
    assert re.search(r"#define\s+SG_STATIC_SCRATCH_BYTES\s+\(16u << 20\)", text) and binding.STATIC_SCRATCH_BYTES == 16 << 20


def test_no_cpu_fallback():
    """Without a CUDA device the product path must fail loudly, not compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    import paper_1309_1599_b200 as sg
    with pytest.raises(sg.SgError):
        sg.SpinGlass(4, 1, 2, 4, [0.6, 0.9, 1.2, 1.6])


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1309_1599_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "sg_oracle" not in text and "import oracle" not in text and "from oracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "sg_oracle.py")).read() + open(os.path.join(ROOT, "oracle", "sg_oracle.c")).read()
    assert "paper_1309_1599_b200" not in otext and "sg_device" not in otext and "sg_kernels" not in otext
    assert not re.search(r"#include\s+\"[^\"]*sg_b200", otext) and "libsg_b200" not in otext


def test_binding_constants_and_struct_layout_match_the_header():
    """The ctypes side restates the header's enums and sg_shape: every enumerator named in include/sg_b200.h has the
    same value in binding.py, and SgShape has the header's fields in the header's order."""
    from paper_1309_1599_b200 import binding
    text = open(os.path.join(ROOT, "include", "sg_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    enums = {}
    for body in re.findall(r"enum\s*\{(.*?)\}", text, flags=re.S):
        nxt = 0
        for item in [t.strip() for t in body.split(",") if t.strip()]:
            name, _, val = [t.strip() for t in item.partition("=")]
            nxt = int(val, 0) if val else nxt
            enums[name] = nxt
            nxt += 1
    for m in re.findall(r"#define\s+(SG_[A-Z_]+)\s+(\d+)", text):
        enums[m[0]] = int(m[1])
    assert enums["SG_EINVAL"] == binding.SG_EINVAL == -1 and enums["SG_ECUDA"] == binding.SG_ECUDA
    checked = 0
    for name, val in enums.items():
        for prefix in ("SG_", "SG_SHAPE_"):
            short = name[len(prefix):] if name.startswith(prefix) else None
            if short and hasattr(binding, short) and isinstance(getattr(binding, short), int):
                assert getattr(binding, short) == val, name
                checked += 1
                break
    assert checked >= 25, checked
    struct = re.search(r"typedef struct \{(.*?)\} sg_shape;", text, flags=re.S).group(1)
    fields = re.findall(r"\b(?:int32_t|uint64_t)\s+([A-Za-z_]+)\s*;", struct)
    assert fields == [f[0] for f in binding.SgShape._fields_]
    assert ctypes.sizeof(binding.SgShape) == 48
