"""Not gpu: the parts of bench.py that need no device -- the byte / op models quoted in DESIGN.md section 5 and the
reference arm (--impl reference times the oracle on a bounded sample and prints the contract's JSON line)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_byte_and_op_models_match_design_md():
    import bench
    import types
    c1 = types.SimpleNamespace(ndim=2, physics=0, r=32, N=1751 * 751, Np=1911 * 911)
    c2 = types.SimpleNamespace(ndim=2, physics=1, r=64, N=2000 * 800, Np=2080 * 880)
    c4 = types.SimpleNamespace(ndim=3, physics=0, r=16, N=512 * 512 * 256, Np=592 * 592 * 336)
    mb = lambda p, T: bench.byte_model(p, T) / 1e6
    assert abs(mb(c1, 0) - 336.6) < 0.1 and abs(mb(c1, 16) - 31.6) < 0.1 and abs(mb(c1, 32) - 21.0) < 0.1
    assert abs(mb(c2, 0) - 819.2) < 0.1 and abs(mb(c2, 16) - 64.0) < 0.1
    assert abs(mb(c4, 0) / 1e3 - 10.95) < 0.01 and abs(mb(c4, 16) / 1e3 - 3.43) < 0.01 and abs(mb(c4, 32) / 1e3 - 3.16) < 0.01
    # ALU model: stencil + update per padded point, r FMAs per probed point
    assert bench.op_model(c1) == 34.0 * c1.Np + 32.0 * c1.N
    assert bench.op_model(c4) == 50.0 * c4.Np + 16.0 * c4.N
    assert bench.kernel_name(c1, 32) == "acoustic2d_stream_kernel" and bench.kernel_name(c4, 0) == "acoustic_step_kernel<3>"


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c0",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["impl"] == "reference" and d["unit"] == "updates/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["n_gpus"] == 1 and d["steps"] == 1 and d["data"] == "synthetic"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("configs[0]")
