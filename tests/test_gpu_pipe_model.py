"""The pipe model DESIGN.md section 6.1 argues from is measured, not assumed: this builds the stand-alone probe
(paper_2409_16053_b200/csrc/probe/pipe_probe.cu) with nvcc and checks, loosely, the three facts the argument needs:
FP64 and FSEL instructions both take about two issue cycles per warp, they overlap when independent, and the
kernel's own PPM4 reconstruction loop stops speeding up with occupancy at about 2 x (FP64 + ALU) cycles."""
import os
import subprocess

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_pipe_probe(tmp_path):
    exe = str(tmp_path / "pipe_probe")
    csrc = os.path.join(ROOT, "paper_2409_16053_b200", "csrc")
    subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-fmad=false", "-I", csrc,
                    "-I", os.path.join(ROOT, "include"), "-o", exe, os.path.join(csrc, "probe", "pipe_probe.cu")], check=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout
    print(out)
    v = {l.split()[0]: float(l.split()[1]) for l in out.splitlines() if not l.startswith("device")}
    for k in ("dfma_cycles_per_warp_instr", "dadd_cycles_per_warp_instr", "dmul_cycles_per_warp_instr", "fsel_cycles_per_warp_instr"):
        assert 1.8 <= v[k] <= 2.8, (k, v[k])
    assert v["dfma_plus_fsel_cycles"] <= 3.2                       # overlap: well under 2 + 2
    assert 3.6 <= v["dfma_plus_2fsel_cycles"] <= 5.2               # the ALU pipe binds: two FSEL
    assert 7.0 <= v["dfma_dependent_latency_cycles"] <= 12.0
    sat, model = v["ppm_recon_loop_cycles_at_30_warps_per_sm"], v["ppm_recon_loop_two_times_fp64_plus_alu"]
    assert 0.85 * model <= sat <= 1.2 * model, (sat, model)
    assert v["ppm_recon_loop_cycles_at_12_warps_per_sm"] <= 1.2 * sat   # 12 warps/SM are already near saturation
