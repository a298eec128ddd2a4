"""CPU-only checks of bench.py's contract: the reference arm (the oracle on the host cores) prints one
JSON line with the agreed keys, and the roofline arithmetic of DESIGN.md section 6 is what bench.py uses."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["metric"] == "electron-steps/s" and j["higher_is_better"] is True
    assert j["value"] > 0 and j["steps"] == 2 and j["warmup"] == 1 and j["dtype"] == "f64"
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] >= 1 and j["cpu_baseline"]["sample"]
    assert j["e2e"] == {"value": j["value"], "unit": j["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in j["config"] and "model" not in j["config"]


def test_reference_arm_under_torchrun_two_ranks():
    """The driver launches both arms the same way; for N > 1 that is torch.distributed.run: rank 0 alone runs the
    oracle and prints the line, the other rank exits 0 without work."""
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29541", os.path.join(ROOT, "bench.py"),
                          "--impl", "reference", "--gpus", "2", "--config", "0", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["n_gpus"] == 2 and j["value"] > 0
    for key in ("metric", "unit", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline", "dtype",
                "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert key in j, key


def test_both_arms_describe_the_workload_identically():
    """`config` is built by one function from the arguments both arms share (no keys that only one arm can fill)."""
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    import workloads as W
    args = argparse.Namespace(step="taylor", gemm_mode="fp32grade")
    cfg = bench.workload_config(W.get_config(3), args)
    assert set(cfg) == {"workload", "ndom_per_gpu", "step", "gemm_mode", "parallelism", "l2"}
    assert "configs[3]" in cfg["workload"] and cfg["ndom_per_gpu"] == 64


def test_algorithmic_counts_match_design():
    sys.path.insert(0, ROOT)
    import bench
    import workloads as W
    c = W.get_config(3)
    a = bench.algorithmic(c)
    elems = 64 * 48 ** 3 * 224
    assert a["elems"] == elems
    assert a["bytes_step"] == elems * 96 + 64 * 48 ** 3 * 20           # 88 B stage passes + 8 B density
    assert abs(a["gemm_flops_step"] - 8 * 4.0 * 64 * 48 ** 3 * 240 * 224) < 1.0   # real beta: 32 N_grid N_proj N_orb per domain
    assert abs(bench.TENSOR_RATIO["fp32grade"] - (1.1 / 2.25) / 3) < 1e-12
    # staged mode: (2 x 3 + 3 x 1 + 3 x 2) / 8 products per MAC on average over the 8 GEMMs of a step
    assert abs(bench.TENSOR_RATIO["staged"] - (1.1 / 2.25) / 1.875) < 1e-12
    assert bench.MODE_NAMES["staged"] == 5


def test_gemm_mode_enum_matches_header():
    """The binding's mode constants are the header's enum values (include/mlmd.h)."""
    import re
    sys.path.insert(0, ROOT)
    from paper_2509_00966_b200 import api
    text = open(os.path.join(ROOT, "include", "mlmd.h")).read()
    enum = dict((m.group(1), int(m.group(2))) for m in re.finditer(r"MLMD_(GEMM_\w+)\s*=\s*(\d+)", text))
    assert enum == {"GEMM_FP32GRADE": 0, "GEMM_FP64": 1, "GEMM_LOWP_BF16": 2, "GEMM_TF32X1": 3, "GEMM_FP32_SIMT": 4,
                    "GEMM_FP32GRADE_STAGED": 5}
    for name, value in enum.items():
        assert getattr(api, name) == value


def test_option_enum_matches_header_and_split_steps_are_accounted():
    """The binding's option keys are the header's enum values, and bench.py's accounting knows the three step forms."""
    import re
    sys.path.insert(0, ROOT)
    from paper_2509_00966_b200 import api
    import bench
    import workloads as W
    text = open(os.path.join(ROOT, "include", "mlmd.h")).read()
    enum = dict((m.group(1), int(m.group(2))) for m in re.finditer(r"^\s+MLMD_(OPT_\w+)\s*=\s*(\d+)", text, re.M))
    assert enum == {"OPT_GRAPH": 0, "OPT_STENCIL": 1, "OPT_GEMM_PATH": 2, "OPT_KICK_NORM": 3, "OPT_FD_ORDER": 4,
                    "OPT_LOCAL_SOLVER": 5, "OPT_COUNT": 6}
    for name, value in enum.items():
        if name != "OPT_COUNT":
            assert getattr(api, name) == value
    c = W.get_config(3)
    elems = 64 * 48 ** 3 * 224
    taylor, split, rich = (bench.algorithmic(c, step=s) for s in ("taylor", "split", "richardson"))
    assert split["gemm_flops_step"] * 2 == taylor["gemm_flops_step"] == rich["gemm_flops_step"] * 2   # two V_NL applications, not four
    assert split["bytes_step"] == taylor["bytes_step"]                       # four Horner stages of h_loc + the density
    assert rich["bytes_step"] == elems * (3 * 16 + 8) + 64 * 48 ** 3 * 20     # three in-place passes + the density
