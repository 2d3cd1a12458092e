"""Host-side pieces of bench.py that need no GPU: the staleness check of profiles/traffic.csv, the
reference arm's JSON line (the oracle on the GPU arm's config) and the OpenMP leg's child process."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SST_CU = os.path.join(ROOT, "paper_2101_11489_b200", "csrc", "sst.cu")


def _bench():
    sys.path.insert(0, ROOT)
    import bench
    return bench


def test_git_blob_sha1_is_what_git_prints():
    bench = _bench()
    want = subprocess.run(["git", "hash-object", SST_CU], capture_output=True, text=True, cwd=ROOT)
    if want.returncode != 0:      # no git here: the definition itself, on a known string
        import hashlib
        assert hashlib.sha1(b"blob 0\0").hexdigest() == "e69de29bb2d1d6434b8b29ae775ad8c2e48c5391"
        return
    assert bench.git_blob_sha1(SST_CU) == want.stdout.strip()


def test_traffic_csv_names_a_blob_and_has_the_three_workloads():
    bench = _bench()
    text = open(os.path.join(ROOT, "profiles", "traffic.csv")).read()
    assert "# sst.cu blob:" in text
    for cfg in (2, 3, 4):
        total, stale = bench.ncu_traffic(cfg)
        assert total and total > 1e8
        assert stale in (True, False)          # True only says: re-capture before quoting roofline.dram


def test_reference_arm_prints_the_gpu_arms_config():
    """`bench.py --impl reference`: the oracle, on the GPU arm's config / metric / unit, each step a
    bounded sample of that workload (here at 3 FEDs so that it takes a second)."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--n-feds", "3", "--ref-events", "2"], capture_output=True, text=True,
                         cwd=ROOT, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads(out.stdout.strip().splitlines()[-1])
    bench = _bench()
    from paper_2101_11489_b200 import synth
    assert d["impl"] == "reference" and d["unit"] == "events/s" and d["higher_is_better"] is True
    assert d["config"] == bench.workload_config(3, 3, bench.N_EVENTS, synth.CONFIGS[3].thresholds[0])
    assert d["config"]["n_events"] == 64 and "first 2 of the workload's 64 events" in d["cpu_baseline"]["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0 and d["value"] > 0


def test_openmp_leg_runs_bound_in_a_child_and_reports_every_shape():
    bench = _bench()
    table, cores, env = bench.time_oracle_omp(1, 3, 2, 1.0)
    assert env == {"OMP_PROC_BIND": "spread,close", "OMP_PLACES": "cores"}
    assert cores == (os.cpu_count() or 1)
    assert len(table) >= 1 and all(t["N"] * t["M"] == cores and t["events_per_s"] > 0 for t in table)
