"""-m gpu: e2e_render_frame_noalloc (the two-kernel render with its scratch in the library's static device array, for callers that
cannot allocate) against the existing path, e2e_render_frame with a caller workspace, on the same inputs.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other tests: the first
call of a process resolves the array's device address, every call rewrites what it reads from the array.
Bar: the frame tolerance of the other GPU tests (|G - R| <= 1e-10 |R| + 1e-14 max(R) per pixel); the two paths launch the same
kernels on the same schedule, so the test also asserts equal bits.
"""
import numpy as np
import pytest

from paper_2008_05858_b200 import workloads as W
from parity_util import assert_frame_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2008_05858_b200 import build, binding
    build.build()
    binding.load()
    return binding


def test_noalloc_render_matches_workspace_render_on_two_calls_in_a_row(B):
    import torch
    # call 1: tiny (BASELINE.json configs[0]); call 2: one RV-sweep frame -- another spectrum, sampling and cell count on the same
    # GPU array, so anything call 1 left behind that call 2 failed to rewrite would show
    scenes = [W.tiny(), W.rv_sweep(10.0)]
    renderers = [B.Renderer(s) for s in scenes]
    try:
        for r in renderers:
            assert r.workspace.numel() <= B.NOALLOC_SCRATCH_BYTES
        want = [r.render().clone() for r in renderers]
        torch.cuda.synchronize()
        got = []
        for r, s in zip(renderers, scenes):                       # two calls in a row, no synchronisation between them
            fr = torch.full((s.ny, s.nx), float("nan"), dtype=torch.float64, device="cuda")
            B.e2e_render_frame_noalloc(r.fmt, r.psf, r.spectra, fr, False)
            got.append(fr)
        torch.cuda.synchronize()
        for g, w, s in zip(got, want, scenes):
            assert w.max().item() > 0
            assert_frame_parity(g.cpu().numpy(), w.cpu().numpy(), "noalloc vs workspace render, " + s.name)
            assert torch.equal(g, w), s.name
        # the same pair again in the other order, and accumulate = 1 on top of a finished frame
        for i in (1, 0):
            fr = torch.full_like(want[i], float("nan"))
            B.e2e_render_frame_noalloc(renderers[i].fmt, renderers[i].psf, renderers[i].spectra, fr, False)
            assert torch.equal(fr, want[i])
        twice = want[0].clone()
        B.e2e_render_frame_noalloc(renderers[0].fmt, renderers[0].psf, renderers[0].spectra, twice, True)
        ref = want[0].clone()
        renderers[0].render(frame=ref, accumulate=True)
        assert torch.equal(twice, ref)
    finally:
        for r in renderers:
            r.close()


def test_noalloc_render_rejects_what_does_not_fit(B):
    import torch
    # 7 orders x 2 fibers of the ESPRESSO-like frame: ~130 000 footprint cells, 136 MB of scratch against the array's 32 MiB
    big = W.espresso_like(n_obj_lines=300, table_dlam=0.01).subset(orders=[0, 1, 2, 40, 41, 83, 84])
    r = B.Renderer(big)
    try:
        assert r.workspace.numel() > B.NOALLOC_SCRATCH_BYTES
        fr = torch.full((big.ny, big.nx), 7.0, dtype=torch.float64, device="cuda")
        with pytest.raises(B.E2EError, match="E2E_ERR_WORKSPACE.*E2E_NOALLOC_SCRATCH_BYTES"):
            B.e2e_render_frame_noalloc(r.fmt, r.psf, r.spectra, fr, False)
        torch.cuda.synchronize()
        assert bool((fr == 7.0).all())                            # nothing was launched
    finally:
        r.close()
    # a tabulated PSF renders with other kernels: no no-allocation form
    t = W.field_psf(base=W.espresso_like(n_obj_lines=300, table_dlam=0.01)).subset(orders=[40])
    r = B.Renderer(t)
    try:
        fr = torch.zeros((t.ny, t.nx), dtype=torch.float64, device="cuda")
        with pytest.raises(B.E2EError, match="E2E_ERR_UNSUPPORTED"):
            B.e2e_render_frame_noalloc(r.fmt, r.psf, r.spectra, fr, False)
    finally:
        r.close()
    # and a pair whose schedule was never built (no e2e_render_workspace_bytes call yet) is refused instead of allocating
    s = W.tiny()
    fmt, psf = B.Format(s), B.Psf(s.psf, s.nx, s.ny)
    try:
        flux = [torch.from_numpy(np.ascontiguousarray(sp.flux, dtype=np.float64)).cuda() for sp in s.spectra]
        desc = B.spectra_array(s.spectra, [f.data_ptr() for f in flux])
        fr = torch.zeros((s.ny, s.nx), dtype=torch.float64, device="cuda")
        with pytest.raises(B.E2EError, match="e2e_render_workspace_bytes"):
            B.e2e_render_frame_noalloc(fmt, psf, desc, fr, False)
        B.e2e_render_workspace_bytes(fmt, psf)
        B.e2e_render_frame_noalloc(fmt, psf, desc, fr, False)
        torch.cuda.synchronize()
        assert fr.max().item() > 0
    finally:
        psf.close()
        fmt.close()
