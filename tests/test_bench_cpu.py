"""Host logic of bench.py that needs no GPU: the algorithmic work per step and the choice of
the roof a dense contraction is held against."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402


def test_c4_algorithmic_work_matches_section_8d():
    """c4: 8 streams x 8192 frames of 8 P^2 flops (P = 1024) and 16 P bytes each plus the (M - 1)-block halo."""
    w = bench.workload_spec("c4")
    flops, byts, _, _ = bench.useful_flops_and_bytes(w)
    assert flops == 8 * 8192 * 8 * 1024 ** 2                     # 549.76 GFLOP
    frames, P, M, S = 8192, 1024, 16, 8
    assert byts == S * ((frames + M - 1) * P * 8 + frames * P * 8) + P * M * 4 or abs(byts - 1.075e9) < 5e6


def test_binding_roof_of_the_dense_contractions():
    """Measured peaks of this pool (MEASURED_PEAKS.json: 1662 TFLOP/s bf16 burst, 6545 GB/s copy): c4 sits on the tensor
    side of the ridge, c2 (N = 256: 192 issued flop per byte against a balance of 254) on the memory side."""
    pk, hbm = 1662.1, 6545.0
    for name, want in (("c4", "tensor"), ("c5", "tensor"), ("c2", "hbm")):
        w = bench.workload_spec(name)
        flops, byts, _, _ = bench.useful_flops_and_bytes(w)
        t_tensor, t_hbm = bench.roof_floors(1.5 * flops, byts, pk, hbm)   # bf16x3 on distinct column pairs: 1.5 issued / useful
        assert ("hbm" if t_hbm > t_tensor else "tensor") == want, (name, t_tensor, t_hbm)
    w = bench.workload_spec("c2")
    flops, byts, _, _ = bench.useful_flops_and_bytes(w)
    t_tensor, t_hbm = bench.roof_floors(1.5 * flops, byts, pk, hbm)
    # per launch; a c2 step is a forward and an inverse launch: 0.082 ms of HBM time against 0.062 ms of tensor time
    assert abs(2 * t_hbm * 1e3 - 0.082) < 0.002 and abs(2 * t_tensor * 1e3 - 0.062) < 0.002
