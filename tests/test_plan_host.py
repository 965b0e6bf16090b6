"""Host logic of the CUDA library (no GPU needed): the library loads, exports every symbol that
include/poisson.h declares, validates arguments, and plans the axis order / work the way the
paper prescribes."""
import ctypes
import re
from fractions import Fraction
from pathlib import Path

import pytest

import paper_1211_5244_b200 as pk

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_1211_5244_b200 import build
    build.build()
    return pk.load_library()


def test_library_exports_every_declared_symbol(lib):
    header = (ROOT / "include" / "poisson.h").read_text()
    declared = set(re.findall(r"POISSON_API[^;]*?\b(poisson_\w+)\s*\(", header))
    assert declared, "no declarations parsed"
    assert declared == set(pk.EXPORTED_SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), f"{name} not exported"
    assert lib.poisson_build_arch().decode() == "sm_100a"


def _golden():
    rows = []
    for line in (ROOT / "tests" / "golden" / "fft_count_ratios.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            name, bx, by, bz, num, den, tn, td = line.split()
            rows.append((name, (int(bx), int(by), int(bz)), Fraction(int(num), int(den)), Fraction(int(tn), int(td))))
    return rows


@pytest.mark.parametrize("name,bc,ratio,transfer", _golden())
def test_fft_count_ratio_matches_paper(lib, name, bc, ratio, transfer):
    """7/12 (free, wire with the periodic axis first), 2/3 (surface, free axis last);
    PAPER.md:23 -- transferred data is 1/8, 1/4, 1/2 of the FFT size."""
    info = pk.poisson_plan_describe(64, 64, 64, bc, pk.FP64)
    assert abs(info.fft_fraction - float(ratio)) < 1e-15
    n = 64 ** 3
    s = info.s[0] * info.s[1] * info.s[2]
    assert Fraction(n, s) == transfer


def test_axis_order_rule(lib):
    """Periodic axes are processed first, free axes last; the R2C axis is never x."""
    for bx in (0, 1):
        for by in (0, 1):
            for bz in (0, 1):
                info = pk.poisson_plan_describe(16, 16, 16, (bx, by, bz), pk.FP64)
                order = list(info.order)
                assert sorted(order) == [0, 1, 2] and order[0] != 0
                bc = (bx, by, bz)
                per = [bc[a] for a in order]
                if bc != (1, 0, 0):  # the one case where "never x first" costs optimality
                    assert per == sorted(per, reverse=True), (bc, order)
    assert list(pk.poisson_plan_describe(16, 16, 16, (0, 0, 0)).order) == [2, 1, 0]
    assert list(pk.poisson_plan_describe(16, 16, 16, (1, 1, 0)).order) == [1, 0, 2]   # surface: z last
    assert list(pk.poisson_plan_describe(16, 16, 16, (0, 0, 1)).order) == [2, 1, 0]   # wire: z first


def test_row_counts_and_bytes_of_the_named_configs(lib):
    """Rows per step (PAPER.md:60-70 with S_x/2+1 -> H on the R2C axis) and B_5 of SURVEY.md 8d."""
    i1 = pk.poisson_plan_describe(128, 128, 128, (0, 0, 0), pk.FP64)
    assert list(i1.s) == [256, 256, 256] and i1.half_len == 129
    assert list(i1.rows) == [128 * 128, 129 * 128, 129 * 256, 129 * 128, 128 * 128]
    assert list(i1.length) == [256] * 5
    assert abs(i1.bytes_total / 1e6 - 506.99) < 0.01
    i0 = pk.poisson_plan_describe(32, 32, 32, (0, 0, 0), pk.FP64)
    assert abs(i0.bytes_total / 1e6 - 8.09) < 0.01
    i2 = pk.poisson_plan_describe(128, 128, 128, (1, 1, 0), pk.FP64)
    assert list(i2.s) == [128, 128, 256] and abs(i2.bytes_total / 1e6 - 186.91) < 0.01
    i3 = pk.poisson_plan_describe(96, 96, 256, (0, 0, 1), pk.FP64)
    assert list(i3.s) == [192, 192, 256] and abs(i3.bytes_total / 1e6 - 304.05) < 0.01
    i4 = pk.poisson_plan_describe(256, 256, 256, (0, 0, 0), pk.FP64)
    assert abs(i4.bytes_total / 1e6 - 4041.21) < 0.01
    i4b = pk.poisson_plan_describe(256, 256, 256, (0, 0, 0), pk.FP32)
    assert abs(i4b.bytes_total / 1e6 - 2020.61) < 0.01
    i4p = pk.poisson_plan_describe(256, 256, 256, (1, 1, 1), pk.FP64)
    assert abs(i4p.bytes_total / 1e6 - 1418.20) < 0.01


def test_argument_validation(lib):
    info = pk.PlanInfo()
    bc = (ctypes.c_int * 3)(0, 0, 0)
    assert lib.poisson_plan_describe(0, 8, 8, bc, 0, ctypes.byref(info)) == 1           # EINVAL: n <= 0
    assert lib.poisson_plan_describe(8, 8, 8, bc, 7, ctypes.byref(info)) == 1           # EINVAL: precision
    assert lib.poisson_plan_describe(8, 8, 8, (ctypes.c_int * 3)(0, 2, 0), 0, ctypes.byref(info)) == 1
    assert lib.poisson_plan_describe(8, 8, 8, bc, 0, None) == 1                          # EINVAL: null
    assert lib.poisson_plan_describe(7, 8, 8, bc, 0, ctypes.byref(info)) == 0           # odd N: planned (any-length kernel)
    assert lib.poisson_plan_describe(8, 8, 14, bc, 0, ctypes.byref(info)) == 0          # S = 28 = 4 * 7: planned
    assert lib.poisson_plan_describe(8, 8, 2049, bc, 0, ctypes.byref(info)) == 2        # EUNSUPPORTED: S = 4098 > 4096
    assert lib.poisson_plan_describe(8, 8, 8, bc, 0, ctypes.byref(info)) == 0
    handle = ctypes.c_void_p(123)
    assert lib.poisson_plan_create(ctypes.byref(handle), 8, 8, 8, bc, -1.0, 0) == 1     # EINVAL: h <= 0
    assert handle.value is None                                                          # *out = NULL on failure
    assert lib.poisson_plan_create(None, 8, 8, 8, bc, 0.1, 0) == 1
    assert lib.poisson_solve(None, None, None, None) == 1
    assert lib.poisson_plan_destroy(None) == 1
    assert b"kernel" in lib.poisson_status_string(4)


def test_plan_create_fails_loudly_without_a_b200(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present; the failure path needs a box without one")
    handle = ctypes.c_void_p()
    st = lib.poisson_plan_create(ctypes.byref(handle), 8, 8, 8, (ctypes.c_int * 3)(0, 0, 0), 0.1, 0)
    assert st == 6 and handle.value is None        # POISSON_EARCH, no fallback
    with pytest.raises(pk.PoissonError):
        pk.PoissonPlan((8, 8, 8), (0, 0, 0), 0.1)


SUPPORTED_LENGTHS = [4, 8, 12, 16, 20, 24, 28, 32, 36, 40, 48, 56, 60, 64, 72, 80, 96, 100, 112, 120, 128, 140, 144, 160, 168, 192,
                     200, 224, 240, 256, 280, 288, 320, 336, 384, 400, 448, 480, 512, 576, 640, 768, 896, 1024]


def test_compiled_lengths_are_those_of_sizes_def():
    text = (ROOT / "paper_1211_5244_b200" / "csrc" / "sizes.def").read_text()
    listed = sorted(int(m) for m in re.findall(r"^PF_SIZE\((\d+),", text, flags=re.M))
    assert listed == SUPPORTED_LENGTHS
    header = (ROOT / "include" / "poisson.h").read_text()
    for v in SUPPORTED_LENGTHS:
        assert re.search(rf"\b{v}\b", header), f"{v} missing from the list in poisson.h"


def test_every_length_is_planned_up_to_the_any_length_limit():
    """DESIGN.md reading 12 ('various grid sizes'): every N >= 1 is planned -- odd N, factors 7, 11, ...,
    primes -- with S = N on a periodic axis and S = 2N on a free one; only a padded length above the
    any-length kernel's limit (4096) is refused with EUNSUPPORTED.  The lengths of csrc/sizes.def keep their compiled
    register-engine kernels (checked on the GPU by the parity sweeps)."""
    for n in list(range(1, 520)) + [521, 769, 1000, 1023, 1025, 2048]:
        for bc_y in (0, 1):
            info = pk.poisson_plan_describe(8, n, 8, (0, bc_y, 0), pk.FP64)
            assert list(info.s) == [16, n * (2 if bc_y == 0 else 1), 16]
            assert info.half_len == info.s[info.order[0]] // 2 + 1 and info.order[0] != 0
        info = pk.poisson_plan_describe(n, 4, 4, (1, 1, 1), pk.FP32)               # odd N_x, periodic: S_x = N_x
        assert list(info.s) == [n, 4, 4]
    for n, bc_z, ok in ((4096, 1, True), (2048, 0, True), (4097, 1, False), (2049, 0, False)):
        try:
            pk.poisson_plan_describe(4, 4, n, (0, 0, bc_z), pk.FP64)
            assert ok
        except pk.PoissonError as e:
            assert e.status == 2 and not ok


def test_half_spectrum_length_and_rows_for_odd_sizes():
    """S_a/2 + 1 outputs are kept by the R2C pass; for odd S_a that is (S_a + 1)/2.  Row counts per step
     for an all-odd surface grid: a = y (periodic), b = x (periodic), c = z (free)."""
    info = pk.poisson_plan_describe(7, 9, 5, (1, 1, 0), pk.FP64)
    assert list(info.s) == [7, 9, 10] and list(info.order) == [1, 0, 2] and info.half_len == 9 // 2 + 1
    assert list(info.rows) == [7 * 5, 5 * 5, 5 * 7, 5 * 5, 7 * 5]
    assert list(info.length) == [9, 7, 10, 7, 9]


def test_reference_arm_of_the_bench_never_loads_the_product_library(lib):
    """`bench.py --impl reference` times the oracle only: its `config` keys come from workloads/ and a restated axis-order
    rule (equal to the planner's for all 8 BCs), and the process must not import the package or map libpoisson_b200.so."""
    import itertools
    import json
    import subprocess
    import sys
    sys.path.insert(0, str(ROOT))
    import bench
    for bc in itertools.product((0, 1), repeat=3):
        assert bench.reference_axis_order(bc) == list(pk.poisson_plan_describe(16, 16, 16, bc, pk.FP64).order)
    code = ("import sys, json, argparse, bench\n"
            "bench.run_reference(argparse.Namespace(config='c0', steps=1, warmup=0, gpus=1))\n"
            "assert 'paper_1211_5244_b200' not in sys.modules\n"
            "assert 'libpoisson_b200' not in open('/proc/self/maps').read()\n")
    r = subprocess.run([sys.executable, "-c", code], cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    info = pk.poisson_plan_describe(32, 32, 32, (0, 0, 0), pk.FP64)
    assert line["impl"] == "reference" and line["config"]["padded_grid"] == list(info.s)
    assert line["config"]["axis_order"] == list(info.order)
