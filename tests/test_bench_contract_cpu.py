"""CPU-only checks of bench.py's contract: the reference arm (the CPU oracle, `--impl reference`) prints the JSON line
the driver expects, with the same `config` object the zmc arm prints, and the roofline table in bench.py matches DESIGN.md."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg1",
                          "--steps", "2", "--warmup", "0"], capture_output=True, text=True, check=True, cwd=ROOT,
                         env=dict(os.environ, RANK="0", WORLD_SIZE="1")).stdout.strip().splitlines()[-1]
    d = json.loads(out)
    assert d["impl"] == "reference" and d["metric"] == "integrand_evals_per_s" and d["unit"] == "evals/s"
    assert d["higher_is_better"] is True and d["steps"] == 2 and d["gpu_launches"] == 0
    assert d["value"] > 0 and d["ms_per_step"] > 0
    assert d["cpu_baseline"]["value"] == d["value"] and d["cpu_baseline"]["cores"] >= 1 and "sample" in d["cpu_baseline"]
    assert d["cpu_baseline"]["single_core"]["value"] > 0
    assert d["e2e"] == {"value": d["value"], "unit": "evals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    import bench
    assert d["config"] == bench.config_of(bench.build_workload("cfg1", 1), 1)       # the zmc arm prints exactly this object


def test_other_ranks_of_the_reference_arm_do_nothing():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg1", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, cwd=ROOT, env=dict(os.environ, RANK="1", WORLD_SIZE="2"))
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_roofline_table_matches_design():
    import bench
    want = {"cfg1": (30, "fp64"), "cfg2": (46, "main(int*2+fp32)"), "cfg3": (84, "main(int*2+fp32)"),
            "cfg4": (127, "main(int*2+fp32)"), "cfg5": (75, "main(int*2+fp32)"), "eq4": (130, "main(int*2+fp32)")}
    for name, (w, bound) in want.items():
        cyc, b, res, no_overlap = bench.w_min(name)
        assert (cyc, b) == (w, bound) and no_overlap >= cyc
    assert abs(bench.PEAK_GLANE - 148 * 128 * 1.965) < 1e-6
    # the physical-unit bound the line headlines (round-3 table; profiles/r03_probe_ncu.md)
    want_pipes = {"cfg1": (30, "fp64"), "cfg2": (39, "issue"), "cfg3": (68, "fma_heavy"), "cfg4": (102.5, "fma_heavy"),
                  "cfg5": (57, "fma_heavy"), "eq4": (96, "fma_heavy")}
    for name, (cyc, unit) in want_pipes.items():
        got, bound, res = bench.pipe_bound(name)
        assert got == cyc and bound.startswith(unit) and got <= bench.w_min(name)[0]     # never looser than the dispatch model
    w = bench.build_workload("eq4_all", 1)
    assert w.G == 10 ** 8 and w.batch_points == 10 ** 6 and bench.config_of(w, 1)["scanned_points"] == 10 ** 8
    w8 = bench.build_workload("cfg5", 8)                                                # weak scaling: 8-fold first list
    assert w8.G == 8 * 10 ** 10 and bench.config_of(w8, 8)["scanned_points"] == 8 * 10 ** 10
