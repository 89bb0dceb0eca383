"""bench.py on the GPU box: the JSON line keeps its contract (keys, types, a roofline fraction that is a fraction) and
`roofline.traffic` is filled, i.e. profiles/x2_traffic.json was captured for the gbe_x2.cu that is checked in."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_keeps_the_contract():
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "3", "--warmup", "3", "--no-cpu-baseline"],
                       cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1  # ONE JSON line
    l = json.loads(lines[0])
    assert l["metric"] == "density_matrix_orbitals_per_s" and l["unit"] == "orbitals/s" and l["higher_is_better"] is True
    assert l["n_gpus"] == 1 and l["steps"] == 3 and l["warmup"] == 3 and l["scaling"] == "weak" and l["vs_baseline"] is None
    assert l["dtype"] == "f64" and l["data"] == "synthetic" and "24576 orbitals" in l["config"]["workload"]
    assert 1e5 < l["value"] < 1e6 and abs(l["value"] - 24576 / (l["ms_per_step"] * 1e-3)) < 1e-6 * l["value"]
    e = l["e2e"]
    assert e["unit"] == l["unit"] and 0 < e["value"] < l["value"]  # the copies are inside its timed region
    assert e["h2d_bytes_per_step"] > 5e7 and e["d2h_bytes_per_step"] > 9e7
    assert l["gpu_launches"] >= 3 * 100  # ~117 of the library's own kernels per step
    c = l["clocks"]
    assert "sm_mhz" in c and "sm_max_mhz" in c and isinstance(c["reasons"], list)  # (values are None without NVML / nvidia-smi)
    r = l["roofline"]
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s" and r["peak"] > 20 and r["achieved"] > 20
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and 0.8 <= r["frac"] <= 1.02
    # traffic comes from the tracked ncu record and is null when gbe_x2.cu changed since it was captured
    assert r["traffic"] is not None and 0.9 <= r["traffic"] / r["algorithmic_bytes_per_launch"] <= 1.1, r.get("traffic_note")


@pytest.mark.parametrize("which", ["packed", "x2"])
def test_timeline_runs_on_the_instrumented_copy(which):
    """bench.py --timeline (profiles/r02_small_m_ncu.md, r02_x2_timeline.md): builds libgbe_stamps.so (-DGBE_STAMPS), loads
    it instead of libgbe.so and prints ordered, plausible stamps; libgbe.so itself exports no stamp reader."""
    import ctypes
    from paper_1603_00937_b200 import binding
    assert not hasattr(ctypes.CDLL(binding.LIB_PATH), "gbe_stamps_x2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--timeline", which], cwd=ROOT, capture_output=True,
                       text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    l = json.loads([x for x in p.stdout.strip().splitlines() if x.startswith("{")][0])
    assert l["timeline"] == which and l["unit"] == "us"
    if which == "packed":
        assert l["sp2_path"] == 3 and l["bins"] >= 148
        for launch in l["launches"]:
            assert 5 < launch["launch_to_launch"] < 200
            for w in launch["waves"]:
                assert 0 < w["setup"] < 20 and 0 < w["copies_issued"] < 20 and 0 < w["units"][0] <= w["units"][1] < 100
                assert 0 < w["slot0_landed_after_release"] <= w["last_slot_landed_after_release"] < 50
    else:
        assert l["tiles"] > 10000 and len(l["launches"]) == 2
        for launch in l["launches"]:
            assert 500 < launch["span"] < 10000 and 0 < launch["epilogue_mean"] < launch["main_loop_mean"] < launch["tile_mean"]
            assert 0.8 < launch["sum_tile_time_over_slots"] / launch["span"] <= 1.0
        assert -50 < l["handover"]["end_to_first_cta_of_next"] < 100
