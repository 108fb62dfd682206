"""The roofline arithmetic bench.py reports (paper_2205_06819_b200/roofline.py) against SURVEY.md sec. 8(d)'s census."""
from paper_2205_06819_b200 import roofline as R


def test_census_matches_the_survey_table():
    c = R.census(3, 9, "fp32")                       # configs 2-4: s = 3, r_k = 9
    assert abs(c["fp32"] - (14 + 6 + 30 + 25 + 4 * 4 * 21 / 9 + 24 / 9)) < 1e-12 and c["mufu"] == 10
    assert abs(c["fp32"] - 115.0) < 0.01             # SURVEY: "Total ~115 FP32, ~10 MUFU -> ~0.90 clk/cell/SM"
    assert abs(R.clocks_per_cell(3, 9, "fp32") - 115.0 / 128) < 1e-3
    c5 = R.census(4, 18, "fp32")                     # config 5: the PSF term is 4 (s+1)(2 r_k + s)/s^2 = 50
    assert abs(c5["fp32"] - (75 + 50 + 1.5)) < 1e-12
    c64 = R.census(3, 9, "fp64")                     # every transcendental expanded to 16 DP instructions
    assert abs(c64["fp64"] - (115.0 + 160)) < 0.01 and c64["fp32"] == 0


def test_roofline_object_fields_and_fraction():
    cells, secs = 16384 * 161604, 11.65e-3
    r = R.roofline(cells, secs, 3, 9, "fp32", sm_mhz_measured=1965.0, traffic=3.4e6)
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert key in r
    assert r["bound"] == "alu" and r["unit"] == "Tinstr/s"
    peak = R.N_SM * 128 * R.sm_max_mhz() * 1e6
    assert abs(r["peak"] * 1e12 / peak - 1) < 1e-12
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9          # the FP32 pipe binds harder than MUFU here
    assert 0.6 < r["frac"] < 0.8                                        # the round-1 measurement of config 3


def test_census_follows_the_component_mask_and_the_tight_count():
    # no bulge (config 4 "2D+H"): the two bulge tables and the lg2 of their argument drop out of the survey's estimate
    c = R.census(3, 9, "fp32", comps=R.DISC1 | R.DISC2 | R.HALO)
    assert abs(c["fp32"] - (14 + 6 + 10 + 25 + 4 * 4 * 21 / 9 + 24 / 9)) < 1e-12 and c["mufu"] == 9
    c = R.census(3, 9, "fp32", comps=R.BULGE | R.DISC1)          # "B+D": one disc
    assert abs(c["fp32"] - (14 + 3 + 30 + 25 + 4 * 4 * 21 / 9 + 24 / 9)) < 1e-12 and c["mufu"] == 9
    # tight census of the tabulated method, four components: 40 2/3 fp32 + 6 MUFU for a2 + a3
    t = R.census(3, 9, "fp32", kind="tight")
    assert abs(t["fp32"] - (40 + 2 / 3 + 4 * 4 * 21 / 9 + 24 / 9)) < 1e-12 and t["mufu"] == 6
    r = R.roofline(16384 * 161604, 11.65e-3, 3, 9, "fp32")
    assert r["frac_tight"] < r["frac"] and abs(r["frac_tight"] / r["frac"] - t["fp32"] / 115.0) < 1e-3
    assert "assumption" in R.roofline(1e9, 1e-2, 3, 9, "fp64")
