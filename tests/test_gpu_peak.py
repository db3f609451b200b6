"""sph_measure_fma_peak: the measured fp32 FMA rate that bench.py reports beside the derived ALU peak of its roofline
(148 SMs x 128 lanes x 2 x 1.965 GHz = 74.4 TFLOP/s).  The bounds are wide on purpose: the test checks
that the helper measures the fp32 pipe (not half of it, not a tensor path), not the clock of the day."""
import pytest

pytestmark = pytest.mark.gpu


def test_measured_fma_peak_is_near_the_derived_one():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2512_09904_b200 import api
    t = api.sph_measure_fma_peak(0, torch.cuda.current_stream().cuda_stream)
    derived = 148 * 128 * 2 * 1.965e9 / 1e12
    assert 0.6 * derived < t < 1.05 * derived, t
