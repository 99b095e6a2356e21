"""Multi-round tiles on EVERY particle.  A tile (256 particles) stages its candidates in rounds of SPH_SE = 1600
slots; at parity sizes almost every tile needs one round, so the paths for two rounds (candidate compaction and slot
renumbering in k_list_compact_sort), for three and more (k_list_sort, the late-candidate ordering of k_cull) and the
round loops of k_density_l / k_pair_l would be checked only on the few tiles of the full-size samples that happen to
need them.  Here a second build of the same sources with SPH_SE = 384 makes every interior tile of the parity cases
need two to five rounds, and the cases -- all fields, neighbour ids of every particle, steps with list reuse and dirty
tiles -- must hold unchanged."""
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SE = 384
CASES = ["tests/test_gpu_rounds.py::test_tiles_do_need_several_rounds_and_all_fields_match",
         "tests/test_gpu_parity.py::test_config0_single_pass_all_fields",
         "tests/test_gpu_parity.py::test_three_tree_levels_and_neighbour_ids",
         "tests/test_gpu_parity.py::test_variable_h_impact_pair_scaled",
         "tests/test_gpu_parity.py::test_skin_lists_give_the_same_single_pass",
         "tests/test_gpu_parity.py::test_fused_step_on_variable_h_two_materials_matches_oracle_stepper",
         "tests/test_gpu_parity.py::test_reused_lists_keep_the_exact_neighbour_sets_over_steps",
         "tests/test_gpu_rungs.py::test_big_step_with_fixed_rungs_matches_the_oracle"]


@pytest.mark.gpu
def test_small_round_build_passes_the_parity_cases(tmp_path):
    sys.path.insert(0, ROOT)
    from paper_2603_19764_b200 import build
    # the candidate pool and the list rows keep the product's sizes (they are stated in units of SPH_SE / per round, and a
    # round of 384 slots pads every chunk's 32 lists four to five times instead of once)
    lib = build.build(out=str(tmp_path / "libsph_se.so"),
                      defines=(f"SPH_SE={SE}", "SPH_POOL_PER_TILE=3200", "SPH_ROWS_DEFAULT=128"))
    env = dict(os.environ, SPH_LIB=lib, SPH_TEST_SE=str(SE))
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-s", "-m", "gpu", *CASES], cwd=ROOT, env=env,
                       capture_output=True, text=True, timeout=1200)
    print(r.stdout[-6000:])
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-2000:]
    assert "passed" in r.stdout and "skipped" not in r.stdout


@pytest.mark.gpu
@pytest.mark.skipif("SPH_TEST_SE" not in os.environ, reason="runs inside test_small_round_build_passes_the_parity_cases")
def test_tiles_do_need_several_rounds_and_all_fields_match():
    from oracle import oracle as O
    from paper_2603_19764_b200 import workloads as W
    from tests import parity_util as U
    se = int(os.environ["SPH_TEST_SE"])
    hist = {}
    for skin in (0.0, 0.1):
        wl = W.elastic_block(14, h_spread=0.25, two_materials=True)
        wl.params.skin = skin
        g = U.gpu_single_pass(wl, split=False, allow_fallback=True)
        ncand, _, flag = g["_sph"].get_tile_stats()
        rounds = (ncand + se - 1) // se
        hist[skin] = np.bincount(rounds).tolist()
        assert flag.sum() == 0 and g["counters"]["list_overflow"] == 0, np.bincount(flag).tolist()   # the list kernels served every tile
        assert (rounds == 2).sum() > 0 and (rounds >= 3).sum() > 0            # both sort kernels were used
        assert (rounds >= 2).mean() > 0.9
        U.compare_single_pass(g, O.single_pass(wl), wl)
        U.neighbor_sets_equal(g["_sph"], wl, mode="brute")
    print("tiles by rounds of", se, "slots:", hist)
