"""fbp_set_trace (include/fbp.h): which launches write %globaltimer marks, and that tracing never changes a byte of the
result.  Traced: the single filter and back-projector launches of fbp_reconstruct / fbp_filter / fbp_backproject.
Never traced: the batch pipeline's per-group launches and fbp_fdk_reconstruct's launches (their grids do not match
the record layout the header documents)."""
import math

import numpy as np
import pytest

from paper_2109_02174_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kind", [pytest.param(2, id="fft"), pytest.param(1, id="direct")])
def test_trace_marks_come_from_the_plain_launches_only(fbp, kind):
    import torch
    k, d, n, b = 24, 95, 64, 8
    ang = I.uniform_angles(k)
    sino = torch.from_numpy(I.random_sinogram(5, b, k, d).astype(np.float32)).cuda()
    with fbp.Plan(list(ang), d, n, dtype="f32", max_batch=b, options={"filter_kind": kind}) as plan:
        want1 = plan.reconstruct(sino[:1]).clone()          # batch 1: sequential path
        want8 = plan.reconstruct(sino).clone()              # batch 8: the batch pipeline (default pipe_min_batch = 8)
        torch.cuda.synchronize()
        info = plan.info()
        assert info["kernels_per_reconstruct"] > 2          # the pipeline is what batch 8 takes
        n_f, n_b = info["filter_ctas"], info["bp_ctas_per_slice"] * b
        marks = torch.zeros(8 * (n_f + n_b) + 64, dtype=torch.int64, device="cuda")
        fbp.fbp_set_trace(plan.handle, marks, marks.numel())
        got1 = plan.reconstruct(sino[:1])
        torch.cuda.synchronize()
        m = marks.cpu().numpy()
        assert m[0] > 0 and m[8 * n_f] > 0                  # filter CTA 0 and back-projector CTA 0 left their start marks
        assert m[4] >= m[0] and m[8 * n_f + 4] >= m[8 * n_f]
        assert torch.equal(got1, want1)                     # the traced instantiation computes the same bytes
        marks.zero_()
        got8 = plan.reconstruct(sino)                       # pipelined: no launch writes marks
        torch.cuda.synchronize()
        assert int(marks.abs().sum()) == 0
        assert torch.equal(got8, want8)
        # cone-beam path on the same plan (2 pi of angles is not needed for this check): never traced
        proj = torch.from_numpy(np.random.default_rng(1).normal(size=(k, 40, d)).astype(np.float32)).cuda()
        plan.fdk_reconstruct(proj, 4.0 * n, 6)
        torch.cuda.synchronize()
        assert int(marks.abs().sum()) == 0
        fbp.fbp_set_trace(plan.handle, None, 0)
