"""bench_probes.cu (measurement only, built by bench.py): the micro-benchmarks behind the measured ALU / L2 peaks of
bench.py's roofline records return sane numbers on a B200."""
import pytest

pytestmark = pytest.mark.gpu


def test_probes_return_sane_peaks():
    import bench
    P = bench.Probes()
    l2 = P.read_bandwidth(48 << 20, 10)
    hbm = P.read_bandwidth(1 << 30, 2)
    assert 1000.0 < hbm < 20000.0 and hbm < l2 < 60000.0      # GB/s: L2-resident reads are faster than HBM reads
    alu = P.alu_lanes_per_clk_per_sm(sm_mhz=1965.0, iters=200)
    assert set(alu) == {"ffma2_3reg", "ffma2_bcast", "fmul2", "fadd2", "ffma", "mufu_rcp"}
    for k, v in alu.items():
        assert 4.0 < v <= 132.0, (k, v)                       # nominal 128 FP32 lanes (16 MUFU lanes) per clock per SM
    assert alu["mufu_rcp"] < 20.0
