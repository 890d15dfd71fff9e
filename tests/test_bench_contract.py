"""CPU-only checks of bench.py's contract: the reference arm (this tier: the oracle on the host
cores) prints one JSON line with the agreed keys, and the clock sampler keeps only the samples of
the timed region."""
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "2",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "particle-steps/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["cpu_baseline"]["value"] == d["value"] == d["e2e"]["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert "workload" in d["config"] and "model" not in d["config"]


def test_reference_arm_other_ranks_do_nothing():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1"], capture_output=True, text=True, timeout=120, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_gpus_flag_must_match_the_launch():
    """--gpus N is never silently ignored: under a launcher it must equal WORLD_SIZE, and without one
    bench.py starts N ranks itself (which fail loudly on a box with fewer devices) instead of printing
    a one-GPU line."""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1"],
                         capture_output=True, text=True, timeout=120, env=env)
    assert out.returncode != 0 and "WORLD_SIZE" in (out.stderr + out.stdout)
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0",
                          "--no-cpu-baseline", "--no-e2e"], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode != 0
    assert '"n_gpus": 1' not in out.stdout


def test_clock_sampler_keeps_the_timed_region_only():
    sys.path.insert(0, ROOT)
    import bench

    class Done:
        def terminate(self): pass
        def wait(self, timeout=None): return 0
        def kill(self): pass

    s = bench.ClockSampler(0)
    s.proc = Done()
    t0 = time.time()

    def line(t, clk, cap):
        ts = time.strftime("%Y/%m/%d %H:%M:%S", time.localtime(t)) + ".%03d" % int((t % 1) * 1000)
        return f"{ts}, 0, {clk}, 1965, 500.0, 0x0, Not Active, Not Active, Not Active, {cap}"

    s.lines = [line(t0 - 5, 300, "Not Active"), line(t0 + 1, 1900, "Active"), line(t0 + 2, 1950, "Not Active"),
               line(t0 + 9, 210, "Not Active"), "garbage"]
    r = s.stop(t0, t0 + 3)
    assert r["samples"] == 2 and r["samples_total"] == 4
    assert r["sm_mhz"] == 1925.0 and r["sm_max_mhz"] == 1965.0 and r["reasons"] == ["sw_power_cap"]
