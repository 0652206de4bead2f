"""Host-side pieces of bench.py (no GPU): the algorithmic work counts it reports against DESIGN.md §6, the derived
FP64 peak, the nvidia-smi sample parser, and the reference arm's JSON line (a short oracle run)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_algorithmic_work_counts_match_the_design_formulas():
    # 3 P 38 + 3 N 17 + 1 FP64 instructions and 3 P 60 + 3 N 34 + 1 flops per system-step (the monitors
    # run on the integer ALU since round 2: no FP64 instruction)
    assert bench.hermite_work(3) == (496, 847)
    assert bench.hermite_work(6)[0] == 2017 and bench.hermite_work(15)[0] == 12736
    for n in range(2, 17):
        P = n * (n - 1) // 2
        assert bench.hermite_work(n) == (3 * P * 38 + 3 * n * 17 + 1, 3 * P * 60 + 3 * n * 34 + 1)


def test_work_models_of_the_other_kernels():
    # the counts quoted there for the tuned shapes
    assert bench.hermite_carry_work(3)[0] == 400 and bench.rkck_work(3)[0] == 604
    assert bench.hermite_adaptive_work(3)[0] == 496 + 62
    assert bench.mvs_work(4)[0] == 3 * 126 + 16 + 3 * 21 == 457 and bench.mvs_work(4, merged=True)[0] == 445
    assert bench.rkck_adaptive_work(3)[0] > bench.rkck_work(3)[0]
    for kind, fn in bench.WORK.items():
        for n in range(2, 17):
            i, f = fn(n)
            assert 0 < i < f < 2 * i, (kind, n)  # every instruction is 1 or 2 flops


def test_traffic_is_read_from_a_committed_profile_or_absent(tmp_path):
    p = tmp_path / "x.txt"
    p.write_text("# header\ndram__bytes_read.sum   24.5 Mbyte\ndram__bytes_write.sum    1.5 Mbyte\n")
    assert abs(bench.profile_traffic(str(p)) - 26.0e6) < 1
    p.write_text("dram__bytes_read.sum 24.5 Mbyte\n")
    assert bench.profile_traffic(str(p)) is None and bench.profile_traffic(str(tmp_path / "missing")) is None


def test_derived_fp64_peak():
    lane, tf = bench.nominal_fp64_peak(148, 1965.0)
    assert abs(lane - 148 * 64 * 1.965e9) < 1 and abs(tf - 37.22496) < 1e-9


def test_clock_sampler_summary_parses_nvidia_smi_rows():
    c = bench.ClockSampler(0)
    c.rows = [["1965", "1965", "120.0", "Not Active", "Not Active", "Not Active", "Not Active"],
              ["1950", "1965", "455.5", "Not Active", "Not Active", "Not Active", "Active"],
              ["1965", "1965", "460.0", "Not Active", "Not Active", "Not Active", "Not Active"],
              ["[N/A]", "x"]]
    s = c.summary()
    assert s["sm_max_mhz"] == 1965.0 and s["sm_mhz"] == 1957.5 and s["reasons"] == ["sw_power_cap"] and s["samples"] == 3
    c.rows = []
    assert c.summary()["sm_mhz"] is None


def test_reference_arm_prints_one_json_line():
    out = subprocess.check_output([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                                   "--warmup", "0"], text=True, env=dict(os.environ, RANK="0"))
    line = json.loads(out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == bench.METRIC and line["unit"] == "system-steps/s"
    assert line["value"] > 1e5 and line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["config"]["workload"] == "hermite_131072x3" and line["higher_is_better"] is True
    # one sample definition for the reference arm and the cpu_baseline leg
    assert line["config"]["sample"] == line["cpu_baseline"]["sample"] and "x 10000 steps" in line["config"]["sample"]
    # under torchrun the other ranks exit 0 without work and without output
    out = subprocess.check_output([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                                   "--warmup", "0"], text=True, env=dict(os.environ, RANK="1", WORLD_SIZE="2"))
    assert out.strip() == ""
