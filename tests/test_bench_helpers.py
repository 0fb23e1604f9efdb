"""Host arithmetic of bench.py's roofline block (no GPU): the line's fractions must be reproducible by hand from
profiles/sweep_counters.csv and MEASURED_PEAKS.json, as DESIGN.md section 7 states them."""
import argparse
import importlib.util
import os

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
bench = importlib.util.module_from_spec(spec)
spec.loader.exec_module(bench)


def test_conflict_free_wavefront_minimum_per_entry_size():
    # four-byte entries at D = 64: 1 load + 5 stores + 2 x (68 x 68 x 4 B / 128 B) / 128 warp-attempts + 1/8
    assert bench.wavefronts_min(6, 1, 1) == pytest.approx(6 + 2 * (68 * 68 * 4 / 128) / 128 + 0.125)
    # two-byte entries (TC=2,2): 3 loads + 3 stores, half the staging; kernel option B = the four-byte variant
    assert bench.wavefronts_min(6, 2, 2) == pytest.approx(6 + 2 * (68 * 68 * 2 / 128) / 128 + 0.125)
    assert bench.wavefronts_min(6, 2, 2, kernel_opt=2) == bench.wavefronts_min(6, 1, 1)
    assert bench.wavefronts_min(8, 1, 1) < bench.wavefronts_min(7, 1, 1)


def test_committed_counters_cover_the_benched_shapes():
    for shape in ((6, 1, 1), (6, 2, 2), (7, 1, 1), (8, 1, 1)):
        c = bench.ncu_counters("sweep_links_kernel", 1 << 16, *shape, 0)
        assert c is not None and c["wavefronts_shared"] > 0 and c["inst_executed"] > 0 and c["dram_bytes"] > 0
        assert os.path.exists(os.path.join(ROOT, c["source"]))
    for log2D in (6, 7):                                      # mixed rates (BASELINE config 3's p, q) are rows of their own
        c = bench.ncu_counters("sweep_links_kernel", 1 << 16, log2D, 1, 1, 0, 0.9, 0.1)
        assert c is not None and c["inst_executed"] > 2 * bench.ncu_counters("sweep_links_kernel", 1 << 16, log2D, 1, 1, 0)["inst_executed"]
    assert bench.ncu_counters("sweep_links_kernel", 1 << 16, 5, 1, 1, 0) is None


def test_roofline_block_is_reproducible_by_hand():
    args = argparse.Namespace(log2D=6, tcx=1, tcy=1, blk=0, kernel=0)
    peaks = {"hbm_gbs": 6543.1, "sm_max_mhz": 1965.0, "src": "measured"}
    L, n_launch, sweep_ms, total_ms = 1 << 16, 128, 128 * 1.75, 128 * 1.75 + 0.5
    rf = bench.roofline_block(args, L, peaks, sweep_ms, total_ms, n_launch, "sweep_links_kernel")
    warp_attempts = L * L / 4 / 32
    peak = 148 * 1965.0e6 / 1e9
    assert rf["bound"] == "smem" and rf["peak"] == pytest.approx(peak)
    assert rf["achieved"] == pytest.approx(bench.wavefronts_min(6, 1, 1) * warp_attempts / 1.75e-3 / 1e9)
    assert rf["frac"] == pytest.approx(rf["achieved"] / peak)
    c = bench.ncu_counters("sweep_links_kernel", L, 6, 1, 1, 0)
    assert rf["wavefronts_per_warp_attempt_measured"] == pytest.approx(c["wavefronts_shared"] / warp_attempts)
    assert rf["pipe_utilisation"] == pytest.approx(c["wavefronts_shared"] / 1.75e-3 / 1e9 / peak)
    assert rf["issue_slots"]["instr_per_attempt_executed"] == pytest.approx(c["inst_executed"] / warp_attempts)
    assert rf["traffic"] == int(c["dram_bytes"])
    assert rf["sweep_share_of_step"] == pytest.approx(sweep_ms / total_ms)
    # L = 2^17 scales the per-launch counters with the domain count
    rf2 = bench.roofline_block(args, 1 << 17, peaks, 4 * sweep_ms, 4 * total_ms, n_launch, "sweep_links_kernel")
    assert rf2["traffic"] == 4 * rf["traffic"] and rf2["frac"] == pytest.approx(rf["frac"])


def test_layout_ceiling_model():
    """Expected wavefronts of a layout that is linear in the site coordinates: a 32-lane access at
    independent random banks costs E[max bank load]; checked against the exact small cases and the known ~3.5 for 32 in 32."""
    assert bench.expected_max_bank_load(1) == 1.0
    # two lanes: 1 + P(same bank) = 1 + 1/32
    assert bench.expected_max_bank_load(2, trials=200000) == pytest.approx(1 + 1 / 32, abs=3e-3)
    assert 3.45 < bench.expected_max_bank_load(32) < 3.62
    lc = bench.wavefronts_expected_linear(6, 1, 1, 0, 0.17)
    assert lc["loads"] == 1 and lc["stores"] == 5
    assert lc["wavefronts_expected_linear"] == pytest.approx(lc["per_load"] + 5 * lc["per_store"] + bench.wavefronts_min(6, 1, 1) - 6)
    assert 12.3 < lc["wavefronts_expected_linear"] < 13.2                  # measured: 13.63 (profiles/sweep_counters.csv)
    args = argparse.Namespace(log2D=6, tcx=1, tcy=1, blk=0, kernel=0)
    peaks = {"hbm_gbs": 6543.1, "sm_max_mhz": 1965.0, "src": "measured"}
    rf = bench.roofline_block(args, 1 << 16, peaks, 128 * 1.75, 128 * 1.75 + 0.5, 128, "sweep_links_kernel", acceptance=0.17)
    assert rf["layout_ceiling"]["frac_of_layout_ceiling"] == pytest.approx(
        rf["frac"] * rf["layout_ceiling"]["wavefronts_expected_linear"] / rf["wavefronts_per_warp_attempt_min"])
