"""-m gpu: bench.py prints ONE JSON line with the keys the driver's contract names, for the
headline mode, the stack mode and (CPU only, rank 0) the reference arm."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
             "scaling", "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches"}


def run(*args, timeout=600):
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                         timeout=timeout, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


@pytest.mark.gpu
def test_headline_line():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    d = run("--steps", "3", "--warmup", "3", "--e2e-steps", "1", "--no-cpu-baseline")
    assert BASE_KEYS | {"clocks"} <= set(d)
    assert d["unit"] == "Mpix/s" and d["steps"] == 3 and d["warmup"] >= 3 and d["n_gpus"] == 1
    assert d["config"]["workload"].startswith("configs[2]") and "model" not in d["config"]
    r = d["roofline"]
    assert r["bound"] in ("hbm", "sm") and 0.3 < r["frac"] < 1.2 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    # both regimes are inside `roofline`, so the driver's record keeps them: burst (idle GPU, boost clocks)
    # cannot be slower than sustained by more than noise, and `bound` is derived from the two, not hard-coded
    assert r["bound_rule"] and 0 < r["kernel_ms_burst"] <= 1.1 * r["kernel_ms"]
    assert r["frac_burst"] >= 0.9 * r["frac"] and r["value_burst"] >= 0.9 * d["value"] and r["ms_per_step_burst"] > 0
    # traffic comes from the tracked ncu capture; null (with the reason) when the kernel sources changed since
    assert r["traffic"] is None or 0.8 < r["traffic"] / r["algorithmic_bytes_per_launch"] < 1.2
    assert r["traffic"] is not None or r["traffic_source"]
    # 4 B per output pixel + 4 B per unique source pixel touched <= 8 B per output pixel
    assert 0.85 * r["upper_bound_bytes_per_launch"] < r["algorithmic_bytes_per_launch"] <= r["upper_bound_bytes_per_launch"]
    assert r["frac"] <= r["frac_upper"] and r["frac_whole_call"] < r["frac"]
    assert d["gpu_launches"] == 3 * d["steps"] and d["value"] > 1e5
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 32 * 2048 * 2048 * 4 == e["d2h_bytes_per_step"] and e["matches_device_path"]
    assert 0 < e["value"] < d["value"]
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}


@pytest.mark.gpu
def test_stack_line():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    d = run("--mode", "stack", "--steps", "3", "--warmup", "3")
    assert BASE_KEYS <= set(d) and d["roofline"]["kernel"].startswith("tiled_stack_kernel")
    assert 20.0 < d["config"]["depth_mean"] <= 32.0


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,extra", [("0", ("--order", "bicubic")), ("1", ()), ("0", ("--src-nx", "254")),
                                       ("4", ("--c4-exposures", "64", "--c4-images", "32"))])
def test_other_configs_print_the_same_contract_line(cfg, extra):
    """bench.py --config {0,1,3,4}: the configs the headline does not time, through the same keys
    (C3 is left to the profiles/ run: its oracle leg alone takes a while)."""
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    d = run("--config", cfg, *extra, "--steps", "3", "--warmup", "3", "--e2e-steps", "1", "--load-seconds", "0.2")
    assert BASE_KEYS | {"clocks"} <= set(d) and d["config"]["workload"].startswith(f"configs[{cfg}]")
    r = d["roofline"]
    assert r["kernel"].startswith("tiled_reproject_kernel") and 0 < r["frac"] < 1.2 and r["kernel_ms"] > 0
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and r["source_pixels_touched"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    e = d["e2e"]
    assert 0 < e["value"] < d["value"] and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    if cfg != "4":
        assert e["max_diff_vs_device_path_dr"] <= 1e-5 and e["mask_diff_vs_device_path"] <= 8
        assert ("<3," if "bicubic" in extra else "<1,") in r["kernel"]
        assert (",0,0>" in r["kernel"]) == ("--src-nx" in extra)            # 254 columns: not staged
    else:
        assert d["exposures_per_s"] > 0 and e["exposures_per_s"] > 0 and d["config"]["distinct_images"] == 32


def test_gpus_n_without_torchrun_starts_its_own_ranks():
    """`python bench.py --gpus 4` with WORLD_SIZE unset re-executes itself under torch.distributed.run
    (one rank per GPU, 127.0.0.1 rendezvous) instead of silently running one rank."""
    sys.path.insert(0, ROOT)
    import bench
    cmd = bench.relaunch_command(["--gpus", "4", "--steps", "2"], 4, port=29511)
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"]
    assert "--nproc-per-node=4" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29511"
    assert cmd[-5:] == [os.path.join(ROOT, "bench.py"), "--gpus", "4", "--steps", "2"]
    free = bench.relaunch_command([], 2)
    assert 1024 < int(free[free.index("--master-port") + 1]) < 65536
    # and the reference arm under it: rank 0 prints the line, the other rank exits 0 without work
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=900, cwd=ROOT,
                         env={k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")})
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1 and lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2


@pytest.mark.gpu
def test_host_multi_line():
    """--mode host_multi on a one-GPU box: two shards, both on device 0 (two pipelines)."""
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    d = run("--mode", "host_multi", "--gpus", "2", "--steps", "1", "--warmup", "1")
    assert d["n_gpus"] == 2 and len(d["config"]["devices"]) == 2
    assert d["reproject_host_multi"]["exposures_per_s"] > 0 and d["stack_host_multi"]["exposures_per_s"] > 0


def test_reference_arm_line():
    """The oracle arm runs on the host cores (no GPU): a bounded sample per step."""
    d = run("--impl", "reference", "--steps", "1", "--warmup", "0", timeout=900)
    assert d["impl"] == "reference" and BASE_KEYS - {"roofline"} <= set(d)      # no kernel, no roofline
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"] and d["gpu_launches"] == 0
