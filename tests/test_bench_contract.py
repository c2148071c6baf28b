"""The bench.py contract that can be checked without a GPU: the reference arm (the oracle on the host
cores) prints one JSON line with the agreed keys, and the GPU arm refuses to run without a device."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, env=None):
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True,
                          cwd=ROOT, env=env, timeout=600)


def test_reference_arm_prints_the_contract_line():
    res = _run(["--impl", "reference", "--gpus", "1", "--steps", "2", "--warmup", "1"])
    assert res.returncode == 0, res.stderr
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "super-droplet-steps/s" and d["unit"] == "sd-steps/s"
    assert d["steps"] == 2 and d["warmup"] == 1 and d["higher_is_better"] is True and d["value"] > 1e5
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["cpu_baseline"]["value"] == d["value"] == d["e2e"]["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert "workload" in d["config"] and "model" not in d["config"]


def test_reference_arm_under_torchrun_env_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    res = _run(["--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"], env=env)
    assert res.returncode == 0 and res.stdout.strip() == ""


def test_gpu_arm_fails_loudly_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    res = _run(["--steps", "1", "--warmup", "1", "--no-e2e", "--no-cpu-baseline"])
    assert res.returncode != 0 and "no CPU fallback" in (res.stderr + res.stdout)


def test_roofline_traffic_comes_from_the_committed_ncu_summaries():
    """bench.py reports roofline.traffic from the committed ncu captures (a profiler is never attached to a timed run)
    and names the file: both summaries exist, parse, and are consistent with the algorithmic 24 B per droplet."""
    sys.path.insert(0, ROOT)
    import bench
    n = 67108864
    fused = bench.ncu_dram_bytes(os.path.join(ROOT, "profiles", bench.TRAFFIC_SOURCES["C5"]))
    general = bench.ncu_dram_bytes(os.path.join(ROOT, "profiles", bench.TRAFFIC_SOURCES["C5s"]))
    assert fused is not None and general is not None
    assert 0.9 < fused / (bench.B_ALG_FUSED_KERNEL * n) < 1.05         # the step kernel moves the algorithmic bytes, once
    assert 1.5 < general / (bench.B_ALG_STEP * n) < 3.0                # shuffled storage: gathers and scattered stores on top
    assert bench.ncu_dram_bytes(os.path.join(ROOT, "profiles", "missing.csv")) is None


def test_roofline_traffic_captures_are_not_older_than_the_kernels_they_describe():
    """roofline.traffic is read from a committed ncu capture, not measured in the run: it goes stale when the kernel
    changes.  The commit that last touched a capture must not be older than the commit that last touched the kernel
    source it describes (needs the git history: skipped in a snapshot without .git, e.g. on the GPU box)."""
    sys.path.insert(0, ROOT)
    import bench

    def last_commit_time(rel):
        res = subprocess.run(["git", "log", "-1", "--format=%ct", "--", rel], capture_output=True, text=True, cwd=ROOT)
        out = res.stdout.strip()
        return int(out) if res.returncode == 0 and out else None

    if not os.path.isdir(os.path.join(ROOT, ".git")) or last_commit_time("bench.py") is None:
        pytest.skip("no git history here")
    for workload, capture in bench.TRAFFIC_SOURCES.items():
        t_cap = last_commit_time(os.path.join("profiles", capture))
        assert t_cap is not None, f"profiles/{capture} is not committed"
        for src in bench.TRAFFIC_KERNEL_SOURCES[workload]:
            t_src = last_commit_time(os.path.join("paper_2101_06318_b200", "csrc", src))
            assert t_src is not None and t_cap >= t_src, (
                f"profiles/{capture} (roofline.traffic of {workload}) is older than the last commit that touched {src}: "
                "re-capture it (command in the .md beside it)")


@pytest.mark.gpu
def test_gpu_arm_prints_the_contract_line():
    """The GPU arm on a small C5-shaped grid (64 x 64 cells): ONE JSON line with the keys of the bench contract --
    throughput, device-timed step, clocks sampled under load, end-to-end through host buffers, launch count, roofline
    of the dominant kernel and the oracle baseline."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    res = _run(["--gpus", "1", "--steps", "6", "--warmup", "3", "--cells", "64", "--e2e-steps", "1"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["metric"] == "super-droplet-steps/s" and d["unit"] == "sd-steps/s" and d["n_gpus"] == 1
    assert d["steps"] == 6 and d["warmup"] == 3 and d["higher_is_better"] is True and d["scaling"] == "weak"
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None
    n = d["config"]["n_sd_per_gpu"]
    assert n == 64 * 64 * 256 and "workload" in d["config"] and "model" not in d["config"]
    assert abs(d["value"] - n * 6 / (d["ms_per_step"] * 6e-3)) <= 1e-6 * d["value"]
    assert d["gpu_launches"] == 2 * 6                      # steady state: sdm_remove_zero + the step kernel
    assert set(("sm_mhz", "sm_max_mhz", "reasons")) <= set(d["clocks"])
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 20 * n and e["d2h_bytes_per_step"] >= 20 * n and 0 < e["value"] < d["value"]
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["peak"] > 1000 and 0 < r["frac"] < 1
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and r["alg_bytes_per_droplet"] == 24.0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] == 1 and c["value"] > 1e5 and "sample" in c and "nproc" in c
