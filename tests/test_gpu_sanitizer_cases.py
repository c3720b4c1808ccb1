"""The small cases chosen for memory- and race-checking (configs 1-2); they are ordinary `-m gpu` parity tests
as well.  `compute-sanitizer` is closed on the GPU pool this was developed on (profiles/r02_sanitizer.md), so no sanitizer log
exists and none is claimed: the memcheck half is done by the library's -DDUALIP_CHECKED build, whose in-kernel bounds
assertions tests/test_gpu_checked_build.py runs these cases against; the racecheck half has no stand-in beyond bit-reproducible
results run to run and across pipeline geometries (tests/test_gpu_parity.py).  What they drive: dualip_create (validation, statistics, tile table), dualip_grad
with x, and a 20-iteration dualip_solve (AGD epilogue, trace buffers) on config 1, its tight companion and config 2 at 60,000
users, through both gradient kernels (TMA-staged k_grad_tma, direct-load k_grad) and both atomic reduction strategies
(per-CTA shared-memory accumulators, RED.ADD.64 to L2) -- the places the round-1 review named: the stage-0 buffer reused as
the epilogue's scratch, 16-byte vector loads past row ends, generic-proxy stores next to bulk copies into the same stage."""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu

if torch.cuda.is_available():
    import paper_2606_07777_b200 as pkg
    from gpu_util import assert_grad_parity, assert_trajectory_parity, from_instance

CASES = [("cfg1", None), ("cfg1-tight", None), ("cfg2", 60_000), ("cfg2-tight", 60_000)]


@pytest.mark.parametrize("name,I", CASES, ids=[c[0] for c in CASES])
@pytest.mark.parametrize("kernel", ["streaming", "direct"])
@pytest.mark.parametrize("red", ["smem", "global"])
def test_grad_with_x_and_short_solve(name, I, kernel, red):
    cfg = synth.get_config(name, I=I) if I else synth.get_config(name)
    inst = synth.generate(cfg)
    po, pg = from_instance(inst, direct_kernel=(kernel == "direct"), reduction={"smem": pkg.RED_SMEM, "global": pkg.RED_GLOBAL}[red])
    info = pg.info()
    assert info.streaming == (1 if kernel == "streaming" else 0)
    assert info.reduction == {"smem": pkg.RED_SMEM, "global": pkg.RED_GLOBAL}[red]
    assert_grad_parity(po, pg, np.zeros(inst.J * inst.m), cfg.gammas[-1], tag=f"{name}/{kernel}/{red}/zero")
    assert_grad_parity(po, pg, synth.probe_lambda(inst, 0, 0.5).numpy(), cfg.gammas[-1], tag=f"{name}/{kernel}/{red}/probe")
    assert_grad_parity(po, pg, synth.probe_lambda(inst, 1, 0.5).numpy(), 0.1, tag=f"{name}/{kernel}/{red}/dense")
    assert_trajectory_parity(po, pg, [10.0 * cfg.gammas[-1], cfg.gammas[-1]], [10, 10], tag=f"{name}/{kernel}/{red}/solve")
    pg.destroy()


def test_jacobi_adaptive_count_row_short_solve():
    """The epilogue's other branches: per-coordinate step, secant step (two-pass finalize), the global-count row."""
    from gpu_util import assert_adaptive_step_parity
    cfg = synth.get_config("cfg2-tight", I=20_000)
    inst = synth.generate(cfg)
    po, pg = from_instance(inst, jacobi=True, adaptive=True, eta_min=1e-5, eta_max=1e-1)
    assert_adaptive_step_parity(po, pg, [1e-2, 1e-3], [10, 10], (1e-5, 1e-1), jacobi=True, tag="sanitizer/adaptive")
    pg.destroy()
    po2, pg2 = from_instance(inst, jacobi=True, count_M=5000.0)
    assert_trajectory_parity(po2, pg2, [1e-2], [10], tag="sanitizer/count", jacobi=True)
    pg2.destroy()
