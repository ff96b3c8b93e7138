"""oracle/flop_counts.json (read by bench.py for the flop side of the roofline) is what the counting build of the oracle
gives today, and the counts behave as the method says they must."""
import json
import os

from oracle import count_flops


def test_stored_counts_are_current_and_consistent():
    stored = json.load(open(count_flops.OUT))["per_zone_stage"]
    fresh = count_flops.count_all()
    assert stored == fresh
    c3, c2, c1 = fresh["3d_plm_hllc_rk2"], fresh["2d_plm_hllc_rk2"], fresh["1d_plm_hllc_rk2"]
    # one sweep per active direction: the 3-D count is about 3/2 of the 2-D one and 3 times the 1-D one (the guard
    # zones' conversions and the 17th faces shift the ratios a little)
    assert 1.4 < c3["flops"] / c2["flops"] < 1.6 and 2.8 < c3["flops"] / c1["flops"] < 3.3
    # square roots: 5 per face with Einfeldt speeds (c_L, c_R, sqrt rho_L, sqrt rho_R, c~), 2 with Davis; 17/16 faces per zone
    # and direction in a 16^3 block, 3 directions
    assert abs(fresh["3d_plm_hllc_rk2"]["sqrt"] - 5 * 3 * 17 / 16) < 1e-3
    assert abs(fresh["3d_plm_hllc_rk2_davis"]["sqrt"] - 2 * 3 * 17 / 16) < 1e-3
    assert abs(fresh["3d_plm_hllc_rk2_8cubed"]["sqrt"] - 5 * 3 * 9 / 8) < 1e-3
    # WENO5 is several times PLM; HLLE and HLLC are within a few per cent of each other
    assert fresh["3d_weno5_hllc_rk3"]["flops"] > 3 * c3["flops"]
    assert abs(fresh["3d_plm_hlle_rk2"]["flops"] / c3["flops"] - 1) < 0.05
