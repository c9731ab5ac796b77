"""CPU tests (``-m "not gpu"``) of the library's host side: the shared object loads and exports every symbol that
include/sparrow.h declares, the host schedule helpers agree with the hand-worked golden values and with the
oracle, workspace sizing, and argument validation (no compute call is made without a GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
from paper_2606_08446_b200 import build as BLD
from paper_2606_08446_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    BLD.build()
    from paper_2606_08446_b200 import binding
    return binding


def test_library_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "sparrow.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sparrow_[a-z_]+)\s*\(", hdr))
    assert {"sparrow_summarize", "sparrow_select", "sparrow_sparse_decode", "sparrow_dense_decode"} <= declared
    lib = ctypes.CDLL(B.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in sparrow.h but not exported"
    assert declared == set(B.EXPORTS), "binding and header disagree"


def test_abi_version_matches_header_and_struct_layout(B):
    """the ABI changed without a version bump.  sparrow_version() == SPARROW_ABI_VERSION of the header == the
    binding's ABI_VERSION (binding.py refuses to import otherwise), and `flags` sits in what used to be padding."""
    hdr = open(os.path.join(ROOT, "include", "sparrow.h")).read()
    ver = int(re.search(r"#define\s+SPARROW_ABI_VERSION\s+(\d+)", hdr).group(1))
    assert B.sparrow_version() == ver == B.ABI_VERSION
    T = B.sparrow_shape_t
    assert ctypes.sizeof(T) == 64 and T.landmark.offset == 32 and T.flags.offset == 36 and T.kv_stride_page.offset == 40
    assert B.sparrow_select_static_bytes() == int(re.search(r"#define\s+SPARROW_SELECT_STATIC_BYTES\s+\((\d+)u << 20\)", hdr).group(1)) << 20


def test_stride_validation(B):
    """sparrow_shape_t kv_stride_*: all zero = packed HND; otherwise 16-byte multiples whose rows do not overlap."""
    shp = B.make_shape(2, 4, 2, 8, 16, kv_layout=(16 * 2 * 128, 128, 2 * 128))
    assert B.sparrow_decode_workspace_bytes(shp, 4) > 0                     # a valid NHD description
    for bad in [(16 * 2 * 128, 128, 128), (16 * 2 * 128 + 4, 128, 256), (0, 128, 256), (4096, 64, 256)]:   # rows overlap / misaligned / zero
        assert B.sparrow_decode_workspace_bytes(B.make_shape(2, 4, 2, 8, 16, kv_layout=bad), 4) == 0


def test_normal_build_carries_no_trace_stamps(B):
    """sparrow_trace_set is declared for every build; only the tracing build (build.py --trace) implements it."""
    lib = ctypes.CDLL(B.LIB_PATH)
    lib.sparrow_trace_set.argtypes = [ctypes.c_void_p]
    assert lib.sparrow_trace_set(None) == -2          # SPARROW_ERR_UNSUPPORTED, and no CUDA call was made
    import subprocess
    sass = subprocess.run(["cuobjdump", "-sass", B.LIB_PATH], capture_output=True, text=True).stdout
    assert "globaltimer" not in sass.lower(), "the normal build reads %globaltimer: trace stamps leaked into it"


def test_built_for_sm100a_with_tensor_and_async_copy_instructions(B):
    import subprocess
    sass = subprocess.run(["cuobjdump", "-sass", B.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in sass
    # tensor-core products (mma.sync -> HMMA, operands via ldmatrix -> LDSM) and the TMA K/V ring of the decode kernel
    # (cp.async.bulk.tensor -> UTMALDG, mbarrier -> SYNCS)
    assert "HMMA" in sass and "LDSM" in sass and "UTMALDG" in sass and "SYNCS" in sass


def _golden():
    for line in open(os.path.join(ROOT, "tests", "golden", "budget_values.txt")):
        line = line.strip()
        if line and not line.startswith("#"):
            c, *v = line.split()
            yield (c, *map(int, v))


@pytest.mark.parametrize("row", list(_golden()), ids=lambda r: f"{r[0]}-L{r[1]}")
def test_host_schedule_matches_hand_worked_values(B, row):
    cfg, L, n_pages, Bt, K, n_forced, k, _ = row
    s = B.make_schedule(W.CONFIGS[cfg]["schedule"])
    assert B.sparrow_budget_tokens(s, L) == Bt
    assert B.sparrow_k_pages(s, L) == K
    assert B.sparrow_forced_count(s, L) == n_forced
    assert B.sparrow_sel_count(s, L) == max(K, n_forced)


def test_host_schedule_agrees_with_oracle_on_random_lengths(B):
    rng = np.random.default_rng(0)
    specs = [W.CONFIGS[c]["schedule"] for c in ("cfg1", "cfg2", "cfg3", "cfg5")]
    specs += [W._sched("table", 40, 300, table_pages=(8, 16, 64, 100, 128), bin_tokens=2048),
              W._sched("dense", 0, 0), W._sched("fixed", 0, 0, fixed_tokens=1), W._sched("fixed", 1000, 5, fixed_tokens=100)]
    for spec in specs:
        for page in (16, 32, 64, 128):                           # Table 4's page sizes
            s, so = B.make_schedule(spec, page_size=page), oracle.Schedule.from_spec(spec)
            lens = [1, 2, 15, 16, 17, 31, 32, 33, 127, 128, 129] + rng.integers(1, 45000, 300 if page == 16 else 80).tolist()
            for L in lens:
                assert B.sparrow_budget_tokens(s, L) == oracle.budget_tokens(so, L, page), (spec, L, page)
                K = oracle.k_pages(so, L, page)
                assert B.sparrow_k_pages(s, L) == K
                F = int(oracle.forced_pages(L, so.sink_tokens, so.local_tokens, page).sum())
                assert B.sparrow_forced_count(s, L) == F
                n_pages = -(-L // page)
                assert B.sparrow_sel_count(s, L) == (n_pages if K >= n_pages else max(K, F))


def test_max_sel_pages_bounds_every_length(B):
    s = B.make_schedule(W.CONFIGS["cfg3"]["schedule"])     # non-monotone budget (R15): peak 200 pages at L = 20480
    assert B.sparrow_max_sel_pages(s, 32768) == 200
    assert B.sparrow_max_sel_pages(s, 8192) == 128
    s5 = B.make_schedule(W.CONFIGS["cfg5"]["schedule"])
    assert B.sparrow_max_sel_pages(s5, 40960) == 128
    sd = B.make_schedule(W._sched("dense", 0, 0))
    assert B.sparrow_max_sel_pages(sd, 1500) == 94


def test_workspace_sizes_and_validation_without_a_gpu(B):
    shp = B.make_shape(64, 16, 8, 1024, 50000)
    assert B.sparrow_select_workspace_bytes(shp) >= 64 * 8 * 4 + 64 * 8 * 1024 * 4
    sparse, dense = B.sparrow_decode_workspace_bytes(shp, 128), B.sparrow_decode_workspace_bytes(shp, 0)
    assert 0 < sparse <= dense
    assert B.sparrow_step_scratch_bytes(shp, 128) > sparse + B.sparrow_select_workspace_bytes(shp)
    # unsupported shapes: status -2 before any pointer is touched; null pointers: -1.  No kernel is launched.
    for bad in (B.make_shape(2, 4, 2, 64, 100, head_dim=64), B.make_shape(2, 4, 2, 64, 100, page_size=48),
                B.make_shape(2, 32, 2, 64, 100), B.make_shape(2, 5, 2, 64, 100)):
        assert B._lib.sparrow_summarize(None, None, None, None, 1, ctypes.byref(bad), None) == -2
        assert B.sparrow_decode_workspace_bytes(bad, 0) == 0
    ok = B.make_shape(2, 4, 2, 64, 100)
    for page in (32, 64, 128):                                     # Table 4's page sizes are supported shapes
        assert B.sparrow_decode_workspace_bytes(B.make_shape(2, 4, 2, 64, 100, page_size=page), 0) > 0
    # the schedule's page size turns B(L) into pages: budget 1024 = 64 / 32 / 16 / 8 pages
    for page, n in ((16, 64), (32, 32), (64, 16), (128, 8)):
        sp = B.make_schedule(W._sched("fixed", 0, 0, fixed_tokens=1024), page_size=page)
        assert B.sparrow_k_pages(sp, 20000) == n and B.sparrow_sel_count(sp, 20000) == n
    assert B.sparrow_k_pages(B.make_schedule(W._sched("fixed", 0, 0, fixed_tokens=1024), page_size=48), 20000) == -1
    assert B._lib.sparrow_summarize(None, None, None, None, 1, ctypes.byref(ok), None) == -1
    assert B._lib.sparrow_summarize(None, None, None, None, 0, ctypes.byref(ok), None) == 0      # empty update: no-op
    s = B.make_schedule(W.CONFIGS["cfg1"]["schedule"])
    assert B._lib.sparrow_select(None, None, None, None, ctypes.byref(s), None, 16, None, None, None, 0, ctypes.byref(ok), None) == -1
    assert B._lib.sparrow_dense_decode(None, None, None, None, None, None, None, 1.0, None, 0, ctypes.byref(ok), None) == -1
    badsched = B.make_schedule(W._sched("linear_frac", 0, 0, f0_ppm=1, f1_ppm=1, L0=5, L1=5))
    assert B.sparrow_budget_tokens(badsched, 100) == -1
    assert "workspace" in B.sparrow_strerror(-3) and B.sparrow_strerror(0) == "ok"


def test_cost_model_helper_matches_the_oracle_restatement():
    """sparrow_cost_model (host helper of the library) against oracle.cost_model, both written from PAPER.md Eq. 2-3 /
    App. F independently; and invalid arguments are refused."""
    import itertools
    import oracle
    from paper_2606_08446_b200 import binding as B
    for L_in, L_out, K, ps, c in itertools.product((0.0, 900.0, 9000.0), (1.0, 700.0, 32000.0), (256.0, 2048.0, 65536.0), (16.0, 128.0), (1.0, 2.0)):
        kw = dict(params=8.0e9, batch_size=2.0, n_samples=8.0, L_in=L_in, L_out=L_out, D=128.0, r=4.0, intensity=295.0,
                  budget_tokens=K, page_size=ps, landmarks_per_page=c)
        got = B.sparrow_cost_model(**kw)
        want = oracle.cost_model(kw["params"], kw["batch_size"], kw["n_samples"], L_in, L_out, 128.0, 4.0, 295.0, K, ps, c=c)
        for k, v in want.items():
            assert abs(got[k] - v) <= 1e-12 * max(1.0, abs(v)), (k, got[k], v, kw)
    with pytest.raises(B.SparrowError):
        B.sparrow_cost_model(params=1.0, batch_size=0.0, n_samples=1.0, L_in=0.0, L_out=1.0, D=128.0, r=1.0, intensity=1.0,
                             budget_tokens=16.0, page_size=16.0, landmarks_per_page=1.0)
