"""-m gpu: every mode of bench.py runs on a small workload and prints one valid JSON line with the keys its contract names
(the measurement tooling of rows d and f1-f4; the numbers themselves are not judged here)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*flags):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *flags], capture_output=True, text=True, timeout=600,
                         cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    return json.loads(out.stdout.strip().splitlines()[-1])


def test_default_step_line(cuda_device):
    d = _run("--workload", "lattice128", "--steps", "3", "--warmup", "3", "--cpu-sample", "2048")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["config"]["workload"] == "lattice128" and d["status"] == 0 and d["gpu_launches"] > 0
    assert d["roofline"]["bound"] == "alu" and 0 < d["roofline"]["frac"] < 1
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1


@pytest.mark.parametrize("flags,mode", [(("--timesteps", "4"), "timestep"), (("--sph", "32", "--steps", "1", "--warmup", "1",
                                                                           "--sph-cpu-sample", "20"), "sph_density"),
                                        (("--pm", "64", "--steps", "2", "--warmup", "1"), "pm_longrange"),
                                        (("--scaling", "let", "--let-domains", "3", "--steps", "2", "--warmup", "1"), "let")])
def test_row_f_modes(cuda_device, flags, mode):
    d = _run("--workload", "lattice128", *flags)
    assert d["mode"] == mode and d["value"] > 0 and d["unit"].startswith("particle")
    if mode == "sph_density":
        assert d["status"] == 0 and abs(d["checks"]["mean_N"] - 32.0) < 1e-3 and d["cpu_baseline"]["max_rel_h_vs_oracle_on_sample"] < 1e-4
    if mode == "pm_longrange":
        assert d["max_abs_acc_difference_between_the_orders_over_rms"] < 1e-3
    if mode == "let":
        assert d["config"]["domains"] == 3 and d["exported_target_copies"] > 0


def test_reference_arm_line(cuda_device):
    d = _run("--impl", "reference", "--workload", "lattice128", "--steps", "1", "--warmup", "1", "--ref-sample", "2048")
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle" and d["extrapolated"] is True
