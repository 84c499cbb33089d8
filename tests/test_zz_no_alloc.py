"""ao_psf_static: the science PSF with its FFT intermediate in the library's static device array (include/ao.h).

Collected last on purpose (pytest -x: a failure here hides nothing).  The entry point must give what the
existing workspace path (ao_psf) gives, on two calls in a row that share the static array, with no workspace lent and
no device memory taken; sizes beyond AO_PSF_STATIC_MAX_BYTES are refused with a clear error.
"""
import numpy as np
import pytest

import oracle
from paper_1608_00386_b200 import inputs
from tests.parity_util import IMAGE_TOL, rel_l2

pytestmark = pytest.mark.gpu

STATIC_MAX_BYTES = 16 << 20          # AO_PSF_STATIC_MAX_BYTES of include/ao.h


def test_psf_static_matches_ao_psf_on_calls_in_a_row():
    import torch
    from paper_1608_00386_b200 import binding
    n_steps, step0 = 3, 5
    cfg = inputs.make_config(3, n_sub=24, screen_n=512, n_steps=n_steps, n_layers=3)     # pupil 288, PSF FFT 1024
    assert cfg.pupil.n * cfg.psf_fft * 8 <= STATIC_MAX_BYTES
    M, sci = cfg.psf_fft, cfg.science_sources()
    geo = binding.Geometry(cfg, workspace_steps=n_steps)
    phase = geo.trace_layers(step0, n_steps, cfg.dt_s)
    want = geo.psf(phase, step0, n_steps, cfg.dt_s)                  # existing path: intermediate in the lent workspace
    # a second, smaller problem on another handle shares the same static array
    cfg_b = inputs.make_config(4, n_sub=8, screen_n=512, n_steps=1, lgs_fft=16, n_layers=2)   # pupil 96, PSF FFT 256
    geo_b = binding.Geometry(cfg_b, workspace_steps=1)
    phase_b = geo_b.trace_layers(0, 1, cfg_b.dt_s)
    want_b = geo_b.psf(phase_b, 0, 1, cfg_b.dt_s)
    torch.cuda.synchronize()
    # from here on: no workspace on either handle, outputs allocated beforehand
    assert geo.lib.ao_set_workspace(geo.handle, None, 0) == 0
    assert geo_b.lib.ao_set_workspace(geo_b.handle, None, 0) == 0
    with pytest.raises(binding.AoError):
        geo.psf(phase, step0, n_steps, cfg.dt_s)                     # the existing path does need the workspace
    d0, d1 = 0, len(sci) - 1
    out0 = torch.full((M, M), float("nan"), dtype=torch.float32, device="cuda")
    out1 = torch.full((M, M), float("nan"), dtype=torch.float32, device="cuda")
    out_b = torch.full((cfg_b.psf_fft, cfg_b.psf_fft), float("nan"), dtype=torch.float32, device="cuda")
    geo.psf_static(d0, phase, n_steps, out0)                         # first call: looks the symbol's address up
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    geo.psf_static(d1, phase, n_steps, out1)                         # two calls in a row, same stream, same array
    geo_b.psf_static(0, phase_b, 1, out_b)                           # another handle, smaller transform, stale contents around it
    geo.psf_static(d0, phase, n_steps, out0, accumulate=True)        # and back: out0 = 2 x PSF
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "ao_psf_static changed the free device memory"
    e0 = rel_l2(out0.cpu().numpy(), 2.0 * want[d0].cpu().numpy())
    e1 = rel_l2(out1.cpu().numpy(), want[d1].cpu().numpy())
    eb = rel_l2(out_b.cpu().numpy(), want_b[0].cpu().numpy())
    assert max(e0, e1, eb) <= IMAGE_TOL, (e0, e1, eb)
    assert torch.equal(out_b, want_b[0])                             # one step, same kernels: the same bits
    # and against the oracle itself (one direction)
    ref = oracle.forward(cfg, step0, n_steps, want_phase=False, want_wfs=False, sources=[sci[d1]])
    assert rel_l2(out1.cpu().numpy(), ref["psf"][sci[d1]]) <= IMAGE_TOL
    assert abs(float(out1.sum()) / n_steps - 1.0) < 1e-4             # Parseval: every PSF sums to 1
    # n_steps = 0 stores zeros; bad arguments are refused
    geo.psf_static(d1, phase, 0, out1)
    torch.cuda.synchronize()
    assert float(out1.abs().max()) == 0.0
    for bad in (-1, len(sci)):
        with pytest.raises(binding.AoError):
            geo.psf_static(bad, phase, 1, out1)


def test_psf_static_refuses_sizes_beyond_its_static_array():
    import torch
    from paper_1608_00386_b200 import binding
    cfg = inputs.make_config(4, n_sub=88, screen_n=512, n_steps=1, lgs_fft=16, n_layers=2)   # pupil 1056, PSF FFT 4096
    assert cfg.pupil.n * cfg.psf_fft * 8 > STATIC_MAX_BYTES
    geo = binding.Geometry(cfg, workspace_steps=1)
    dummy = torch.zeros(16, dtype=torch.float32, device="cuda")      # never touched: the size check comes first
    with pytest.raises(binding.AoError) as err:
        geo.psf_static(0, dummy, 1, dummy)
    assert err.value.status == 3                                     # AO_ERR_UNSUPPORTED
    assert "AO_PSF_STATIC_MAX_BYTES" in str(err.value) and str(cfg.pupil.n * cfg.psf_fft * 8) in str(err.value)
    assert np.all(dummy.cpu().numpy() == 0.0)


def test_psf_static_replays_from_a_cuda_graph():
    """The reason the entry point exists: a call captured into a CUDA graph (where cudaMalloc is forbidden) replays with
    the same result as the workspace path, for two different phase buffers copied into the captured input."""
    import torch
    from paper_1608_00386_b200 import binding
    cfg = inputs.make_config(4, n_sub=8, screen_n=512, n_steps=2, lgs_fft=16, n_layers=2)   # pupil 96, PSF FFT 256
    M = cfg.psf_fft
    geo = binding.Geometry(cfg, workspace_steps=2)
    ph_a = geo.trace_layers(0, 2, cfg.dt_s)
    ph_b = geo.trace_layers(40, 2, cfg.dt_s)
    want_a = geo.psf(ph_a, 0, 2, cfg.dt_s)[0].clone()
    want_b = geo.psf(ph_b, 40, 2, cfg.dt_s)[0].clone()
    buf = ph_a.clone()
    out = torch.zeros((M, M), dtype=torch.float32, device="cuda")
    geo.psf_static(0, buf, 2, out)                                   # warm-up outside the capture (symbol address, attributes)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        geo.psf_static(0, buf, 2, out)
    for ph, want in ((ph_b, want_b), (ph_a, want_a)):
        buf.copy_(ph)
        out.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        assert rel_l2(out.cpu().numpy(), want.cpu().numpy()) <= IMAGE_TOL
