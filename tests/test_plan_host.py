"""Host logic of the resident engine, no GPU: the tiling planner and the halo-exchange pattern (cav_plan_check, include/cavity_debug.h).

Every unit of four grid points that a tile fetches from its ring must be stored by exactly one tile (the owner of those
points), every stored unit must be fetched by some neighbour, and every tile must fit its thread grid: a mismatch would
leave a tile waiting forever for data nobody sends ("Halo exchange").  The exchange itself is checked
bit for bit against the oracle on the GPU (tests/test_gpu_parity.py); this covers the sizes those tests do not reach."""
import pytest

from paper_0809_3098_b200 import binding

SIZES = [2, 31, 32, 33, 64, 65, 96, 100, 127, 128, 129, 130, 131, 219, 256, 299, 300, 511, 512, 513, 777, 1000, 1022, 1023, 1024, 1025,
         1500, 2047, 2048]


@pytest.mark.parametrize("sweep", ["redblack", "compact9"])
def test_exchange_pattern_is_consistent_for_every_plan(sweep):
    seen_multi = 0
    for N in SIZES:
        for T in (0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10):
            rc, plan, counts = binding.plan_check(N, sweep, T)
            if rc == -4:                 # no resident plan for this forced T (or grid too large for 148 tiles)
                continue
            assert rc == 0, (N, sweep, T, plan, counts)
            assert counts["unmatched"] == 0 and counts["unfetched"] == 0 and counts["misfit"] == 0
            assert plan["ntx"] * plan["nty"] <= 148
            if plan["ntx"] * plan["nty"] > 1:
                seen_multi += 1
                assert counts["fetched"] >= counts["stored"] > 0          # a border unit is fetched by up to three neighbours
                assert plan["halo"] == (4 if sweep == "compact9" else 2) * plan["T"]
                if T:
                    assert plan["T"] == T
                # the cores cover the grid: rows [0, nty CH), columns [0, ntx CW + 1), CW a multiple of four when split in x
                if plan["EB"] == 0:
                    assert plan["nty"] * plan["CH"] >= N + 1 and (plan["nty"] - 1) * plan["CH"] < N + 1
                else:      # first row of tiles CH + EB rows, the last row the rest (more than the halo, at most 96 - halo - 5)
                    assert 0 < plan["EB"] <= plan["halo"]
                    last = N + 1 - plan["EB"] - (plan["nty"] - 1) * plan["CH"]
                    assert plan["halo"] < last <= 6 * plan["warps"] - plan["halo"] - 5
                if plan["ntx"] > 1:
                    assert plan["CW"] % 4 == 0 and plan["ntx"] * plan["CW"] >= N and (plan["ntx"] - 1) * plan["CW"] < N
            else:
                assert counts["fetched"] == 0 and counts["stored"] == 0
    assert seen_multi > 50


def test_plan_of_the_headline_config_and_device_limits():
    rc, plan, counts = binding.plan_check(1024, "redblack")
    assert rc == 0 and plan["ntx"] * plan["nty"] <= 148 and plan["warps"] == 16 and plan["T"] >= 4
    # fewer multiprocessors: fewer, not larger, tiles are impossible (a tile is at most 128 x 96 points) -> no plan
    assert binding.plan_check(1024, "redblack", 0, sms=64)[0] == -4
    # less shared memory than a tile image needs -> no plan
    assert binding.plan_check(1024, "redblack", 0, smem_bytes=48 * 1024)[0] == -4
    # bad arguments
    assert binding.plan_check(1, "redblack")[0] == -1
    assert binding.lib().cav_plan_check(64, 1, 0, 148, 232448, None, None) == -1      # Jacobi has no resident plan kind
