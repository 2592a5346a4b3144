"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol that
include/mfh.h declares, host-side argument checking, and the analytic planner's arithmetic
against the sizes the paper prints."""
import ctypes
import os
import re

import pytest

from paper_2606_31598_b200 import binding as mfh

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "mfh.h")).read()
    declared = sorted(set(re.findall(r"MFH_API\s+(?:const\s+)?\w+\*?\s+(mfh_\w+)\s*\(", hdr)))
    assert declared == sorted(mfh.SYMBOLS)
    L = mfh.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_31598_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "mfh_oracle" not in src, f


@pytest.mark.parametrize("D,B", [(100, 32), (4096, 48), (4096, 8192), (16, 16), (4096, 96)])
def test_create_rejects_bad_sizes(D, B):
    with pytest.raises(mfh.MfhError) as e:
        mfh.Hamiltonian(D, B)
    assert e.value.code == mfh.MFH_ERR_INVALID_ARG


def test_create_rejects_bad_enums_and_lambda():
    import ctypes
    L = mfh.lib()
    h = ctypes.c_void_p()
    assert L.mfh_create(ctypes.byref(h), 4096, 512, 1, 7, 1.0, 0, 0) == mfh.MFH_ERR_INVALID_ARG
    assert L.mfh_create(ctypes.byref(h), 4096, 512, 1, 0, 1.0, 5, 0) == mfh.MFH_ERR_INVALID_ARG
    assert L.mfh_create(ctypes.byref(h), 4096, 512, 1, 0, float("nan"), 0, 0) == mfh.MFH_ERR_INVALID_ARG
    assert L.mfh_create(None, 4096, 512, 1, 0, 1.0, 0, 0) == mfh.MFH_ERR_INVALID_ARG
    assert L.mfh_destroy(None) == mfh.MFH_OK


def test_bad_state_before_plan():
    h = mfh.Hamiltonian(4096, 512, 1234)
    with pytest.raises(mfh.MfhError) as e:
        h.get_plan()
    assert e.value.code == mfh.MFH_ERR_BAD_STATE
    import ctypes
    L = mfh.lib()
    rc = L.mfh_apply(h._h, ctypes.c_void_p(16), ctypes.c_void_p(32), 1, None, None)
    assert rc == mfh.MFH_ERR_BAD_STATE
    assert L.mfh_apply(h._h, None, ctypes.c_void_p(32), 1, None, None) == mfh.MFH_ERR_INVALID_ARG
    h.destroy()


# ---- planner arithmetic (Algorithm 1; Eq. 13-18) --------------------------------------------

def test_planner_memory_model_matches_paper_sizes():
    # a complex64 dense operator of dimension 2^18 needs 8*(2^18)^2 = 2^39 B (512 GiB);
    # 65536^2 * 8 = 32 GiB; a 4096^2 complex64 block = 128 MiB.
    r = mfh.plan_analytic(262144, "c64", 1, "procedural", 4096, 1, 180 * 10**9)
    assert r["dense_bytes"] == 2**39
    r = mfh.plan_analytic(65536, "c64", 1, "full", 4096, 1000, 180 * 10**9)
    ch = r["chosen"]
    assert ch["mode"] == "full" and ch["cache_bytes"] == 32 * 2**30
    assert ch["cached_blocks"] == 16 * 16 and ch["cache_bytes"] / ch["cached_blocks"] == 128 * 2**20


def test_planner_flops_formula():
    # Eq. 13: F_mv = 8 n_op D_out D_in R; the paper's 2.749e11 = 2 * 4 * 65536^2 * 8.
    r = mfh.plan_analytic(65536, "c64", 4, "procedural", 4096, 1, 180 * 10**9)
    assert r["chosen"]["flops_per_apply"] == pytest.approx(8 * 65536**2 * 4, rel=1e-5)
    assert 2 * r["chosen"]["flops_per_apply"] == pytest.approx(2.749e11, rel=1e-3)


def test_planner_rejects_what_does_not_fit():
    # C4: the dense matrix is 1.1 TB, full cache can never fit (Eq. 18) -> OUT_OF_MEMORY when forced
    with pytest.raises(mfh.MfhError) as e:
        mfh.plan_analytic(262144, "c128", 1, "full", 4096, 10, 180 * 10**9)
    assert e.value.code == mfh.MFH_ERR_OUT_OF_MEMORY
    r = mfh.plan_analytic(262144, "c128", 1, "auto", 4096, 10, 180 * 10**9)
    assert r["chosen"]["feasible"] and r["chosen"]["mode"] in ("procedural", "partial", "pairs")
    assert r["chosen"]["total_bytes"] <= 0.9 * 180e9


def test_planner_c2_full_cache_size_and_c5_partial_budget():
    r = mfh.plan_analytic(65536, "c128", 1, "full", 2048, 100, 180 * 10**9)
    ch = r["chosen"]
    assert ch["cache_bytes"] == 65536**2 * 16 and ch["cached_blocks"] == 1024   # 68.7 GB, 32x32 blocks
    # C5: 275 GB total, about 150 GB cached (Eq. 27: P_cache = floor(M_cache / (B_c b^2)), row balanced)
    r = mfh.plan_analytic(131072, "c128", 1, "partial", 4096, 151, int(150e9 / 0.9))
    ch = r["chosen"]
    assert ch["mode"] == "partial" and ch["total_bytes"] <= 150e9
    assert ch["cached_blocks"] == ch["cached_per_row"] * 32
    assert ch["cache_bytes"] + 32 * 4096**2 * 16 + ch["work_bytes"] > 150e9 * 0.97   # one more per row would not fit


def test_planner_enumerates_block_sizes_and_ranks_feasible_first():
    r = mfh.plan_analytic(65536, "c128", 1, "auto", 0, 100, 180 * 10**9)
    Bs = {c["B"] for c in r["candidates"]}
    assert {4096, 2048, 1024, 512} <= Bs
    flags = [c["feasible"] for c in r["candidates"]]
    assert flags == sorted(flags, reverse=True)
    feas = [c["model_job_s"] for c in r["candidates"] if c["feasible"]]
    assert feas == sorted(feas)


def test_pairs_mode_and_pipe_rate_arguments():
    # Hermitian pair cache in the analytic planner: half the bytes of the full cache, all entries covered
    r = mfh.plan_analytic(65536, "c128", 1, "pairs", 2048, 100, 180 * 10**9)
    ch = r["chosen"]
    assert ch["mode"] == "pairs" and ch["cached_fraction"] == 1.0
    assert ch["cached_blocks"] == 32 * 33 // 2 and ch["cache_bytes"] == 528 * 2048**2 * 16
    # C5: the whole operator fits the 150 GB budget as pairs (141.7 GB), not as full blocks (275 GB)
    r = mfh.plan_analytic(131072, "c128", 1, "pairs", 4096, 151, int(150e9 / 0.9))
    assert r["chosen"]["cached_fraction"] == 1.0 and r["chosen"]["total_bytes"] <= 150e9
    # k-vector plans: cached blocks need B % 128 == 0 (tensor-core kernel for complex64, FP64 kernel for
    # complex128); never pairs
    r = mfh.plan_analytic(32768, "c64", 16, "full", 1024, 100, 180 * 10**9)
    assert r["chosen"]["feasible"] and r["chosen"]["cache_bytes"] == 32768**2 * 8
    r = mfh.plan_analytic(32768, "c128", 16, "full", 1024, 100, 180 * 10**9)
    assert r["chosen"]["feasible"] and r["chosen"]["cache_bytes"] == 32768**2 * 16
    for dtype, B, mode in [("c128", 96, "full"), ("c64", 96, "full"), ("c128", 1024, "pairs")]:
        with pytest.raises(mfh.MfhError) as e:
            mfh.plan_analytic(3072 * 8, dtype, 16, mode, B, 100, 180 * 10**9)
        assert e.value.code == mfh.MFH_ERR_OUT_OF_MEMORY
    # measurement export: argument errors come before any device work
    L = mfh.lib()
    out = ctypes.c_double(0.0)
    assert L.mfh_debug_pipe_rates(99, ctypes.byref(out), None) == mfh.MFH_ERR_INVALID_ARG
    assert L.mfh_debug_pipe_rates(0, None, None) == mfh.MFH_ERR_INVALID_ARG


def test_auto_enumeration_is_fast_at_the_largest_sizes():
    """B = 0 enumerates block sizes; the candidate search must stay interactive at D = 2^18 (it once built
    N_blk^2 tables for N_blk = 8192 thousands of times)."""
    import time
    t0 = time.time()
    for D, dtype, k, free, n in [(262144, "c128", 1, 180e9, 10), (131072, "c128", 1, 150e9 / 0.9, 151),
                                 (32768, "c64", 16, 180e9, 100)]:
        rec = mfh.plan_analytic(D, dtype, k=k, n_applies_hint=n, hbm_free_bytes=int(free))
        assert rec["chosen"]["feasible"] and all(c["n_blk"] <= 256 for c in rec["candidates"])
    assert time.time() - t0 < 20.0
    # C5 inside its 150 GB budget: the Hermitian pair cache holds the whole operator, AUTO prefers it to partial
    rec = mfh.plan_analytic(131072, "c128", k=1, n_applies_hint=151, hbm_free_bytes=int(150e9 / 0.9))
    assert rec["chosen"]["mode"] == "pairs" and rec["chosen"]["cached_fraction"] == 1.0


def test_node_planner_reproduces_the_papers_hybrid_plan():
    """P:765-779 and Fig. 1: eight 43.97 GiB GPUs, two dense complex64 bath operators of d_B = 65536 on R = 4
    columns, 20 coupling values -> full-cache hybrid plan with row-group size 2: gpu groups [[0,1],...,[6,7]], 32 GiB
    of operator storage per GPU, five waves; row-group size 4 needs ten waves; one GPU cannot hold 64 GiB."""
    from paper_2606_31598_b200.distributed import row_groups, task_waves
    GiB = 2**30
    rec = mfh.plan_node_analytic(65536, "c64", 4, 2, 20, 8, int(43.97 * GiB), mode="full", B=4096, scheme="rows",
                                 n_applies_per_task=1000)
    by = {r["p_row"]: r for r in rec["row_groups"]}
    assert sorted(by) == [1, 2, 4, 8]
    assert not by[1]["feasible"] and by[1]["operator_bytes_per_gpu"] == 64 * GiB          # Eq. 15, Eq. 18
    ch = rec["chosen"]
    assert ch["p_row"] == 2 and ch["groups"] == 4 and ch["waves"] == 5 and ch["strategy"] == "hybrid"
    assert ch["operator_bytes_per_gpu"] == 32 * GiB                                       # "32 GiB ... per GPU"
    assert ch["total_bytes_per_gpu"] <= 32.2 * GiB                                        # "32.1 GiB total"
    assert rec["flops_per_apply"] == pytest.approx(2.749e11, rel=1e-3)                    # "2 d_S d_R^2 8"
    assert by[4]["waves"] == 10 and by[8]["waves"] == 20 and by[8]["strategy"] == "row-parallel"
    assert by[4]["model_apply_s"] < ch["model_apply_s"] and by[4]["score_s"] > ch["score_s"]   # Fig. 1 A2
    # the printed score: five waves of the measured 0.104089 s
    assert len(task_waves(20, ch["groups"])) == 5 and 5 * 0.104089 == pytest.approx(0.520447, abs=3e-6)
    assert row_groups(8, 2) == [[0, 1], [2, 3], [4, 5], [6, 7]]                            # "gpu groups = ..."
    # with the mode left open the planner still prefers the fully cached row groups of two
    auto = mfh.plan_node_analytic(65536, "c64", 4, 2, 20, 8, int(43.97 * GiB), n_applies_per_task=1000, scheme="rows")
    assert auto["chosen"]["p_row"] == 2 and auto["chosen"]["mode"] == "full"
    # one B200 holds both operators: with 16 tasks on eight GPUs parameter-parallel execution wins (two full waves);
    # with the paper's 20 tasks its third wave is half empty and row groups of two (five full waves) stay ahead
    b200 = mfh.plan_node_analytic(65536, "c64", 4, 2, 16, 8, 180 * 10**9, n_applies_per_task=1000)
    assert b200["chosen"]["p_row"] == 1 and b200["chosen"]["waves"] == 2 and b200["chosen"]["strategy"] == "parameter-parallel"
    b200 = mfh.plan_node_analytic(65536, "c64", 4, 2, 20, 8, 180 * 10**9, n_applies_per_task=1000)
    assert b200["row_groups"][0]["feasible"] and b200["row_groups"][0]["waves"] == 3 and b200["chosen"]["p_row"] == 2
    with pytest.raises(mfh.MfhError) as e:
        mfh.plan_node_analytic(65536, "c64", 4, 2, 20, 8, 2 * GiB, mode="full", B=4096)
    assert e.value.code == mfh.MFH_ERR_OUT_OF_MEMORY
    with pytest.raises(mfh.MfhError) as e:
        mfh.plan_node_analytic(65536, "c64", 4, 0, 20, 8, 40 * GiB)
    assert e.value.code == mfh.MFH_ERR_INVALID_ARG


def test_task_waves_cover_every_task_once():
    from paper_2606_31598_b200.distributed import my_tasks, row_groups, task_waves
    for n_tasks, C in [(20, 4), (20, 8), (7, 3), (1, 4), (16, 16)]:
        waves = task_waves(n_tasks, C)
        assert len(waves) == -(-n_tasks // C)
        flat = [t for w in waves for (_, t) in w]
        assert flat == list(range(n_tasks))
        assert all(len({g for (g, _) in w}) == len(w) for w in waves)          # a group runs one task per wave
        assert sorted(t for g in range(C) for t in my_tasks(n_tasks, g, C)) == list(range(n_tasks))
    with pytest.raises(ValueError):
        row_groups(8, 3)


def test_partitioned_handle_needs_a_fixed_block_size():
    """Block ownership is defined in block indices: mfh_plan refuses B = 0 on a partitioned handle before any device
    work (ranks picking different B would own sets that do not tile H)."""
    import ctypes
    L = mfh.lib()
    h = mfh.Hamiltonian(4096, 0, 1234)
    h.set_partition(0, 2, "pairs")
    buf = ctypes.create_string_buffer(64)
    assert L.mfh_plan(h._h, mfh.MFH_MODE_PROCEDURAL, 1, 1, 0, 0, None, buf, 64) == mfh.MFH_ERR_INVALID_ARG
    assert b"same B" in L.mfh_last_error()
    h.destroy()


def test_bessel_table_of_the_chebyshev_driver_against_scipy():
    """mfh_chebyshev's Jacobi-Anger coefficients (Miller recurrence) at small, moderate and LARGE arguments; the large
    ones are where std::cyl_bessel_j breaks down (x > 1000 at high order)."""
    import numpy as np
    from scipy.special import jv
    for x in (0.0, 0.3, 7.5, 105.0, 713.0, 1001.0, 2000.0):
        l_max = int(x + 80 + 12 * np.cbrt(x))
        J = mfh.bessel_j_table(x, l_max)
        ref = jv(np.arange(l_max + 1), x)
        assert np.all(np.isfinite(J)) and np.max(np.abs(J - ref)) < 1e-13, x
        assert abs(J[0] ** 2 + 2.0 * np.sum(J[1:] ** 2) - 1.0) < 1e-12      # sum rule J_0^2 + 2 sum J_l^2 = 1
    assert mfh.bessel_j_table(1001.0, 500)[500] == pytest.approx(-0.0270214558893, rel=1e-9)   # libstdc++ gave -4.2e33
    with pytest.raises(mfh.MfhError):
        mfh.bessel_j_table(-1.0, 10)
