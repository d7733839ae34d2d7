"""glisse_planet_log_static (include/glisse.h): the planet log for callers that may not allocate — the
planet-history kernel's Jacobi-state scratch in a file-scope static __device__ array (csrc/planets.cu), the log
written straight into the caller's device buffer — against the existing glisse_planet_log (scratch and staging
from cudaMalloc).  Both launch the same kernel, so the records must agree to the last bit; the planet log's own
tolerance against the oracle (tests/test_gpu_parity.py: PLANET_TOL) is what the existing path is held to.

Collected last on purpose (file name): the suite runs with pytest -x, and a failure here must not hide the
parity tests.  Passes alone in a fresh process and after the other tests: it shares no state with them but the
library's static scratch, which no other entry point touches.
"""
import numpy as np
import pytest

from paper_2011_03484_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gl():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2011_03484_b200 import binding
    binding.lib()
    return binding


def test_planet_log_without_allocation_matches_the_allocating_path(gl):
    import torch
    # two calls in a row that share the scratch: a long log first (N_p = 8, config 4's planets), then a shorter
    # one of another system (N_p = 4) whose records land on what the first call left behind; then the first again
    calls = ((inputs.config(4, 64), 1500), (inputs.config(1, 64), 700), (inputs.config(4, 64), 1500))
    for w, n_steps in calls:
        S = gl.GlisseSim.from_workload(w, chunk_steps=256)
        S.advance(300)                                   # not at the origin of the planet clock
        stride = gl.log_stride(w.n_planets)
        want = S.planet_log(n_steps)                     # the existing path (allocates)
        out = torch.full((n_steps + 1, stride), float("nan"), dtype=torch.float64, device="cuda")
        S.planet_log_static(n_steps, out)
        got = out.cpu().numpy()
        assert np.array_equal(got, want)                 # the same kernel: bit for bit
        # a second call on the same sim, straight after: the simulation was not changed, the scratch is reused
        out2 = torch.full((n_steps + 1, stride), float("nan"), dtype=torch.float64, device="cuda")
        S.planet_log_static(n_steps, out2)
        assert np.array_equal(out2.cpu().numpy(), want)
        # ... and the sim goes on as if nothing had happened
        S.advance(50)
        q, v = S.read_planets()
        S.close()
        T = gl.GlisseSim.from_workload(w, chunk_steps=256)
        T.advance(350)
        q0, v0 = T.read_planets()
        T.close()
        assert np.array_equal(q, q0) and np.array_equal(v, v0)


def test_planet_log_without_allocation_refuses_what_it_cannot_hold(gl):
    import torch
    assert gl.planet_log_static_limit(4) == (1 << 18) // 24 - 1 == 10921
    assert gl.planet_log_static_limit(8) == 5460 and gl.planet_log_static_limit(32) == 1364
    assert gl.planet_log_static_limit(33) < 0
    w = inputs.config(1, 64)
    S = gl.GlisseSim.from_workload(w, chunk_steps=256)
    stride = gl.log_stride(w.n_planets)
    lim = gl.planet_log_static_limit(w.n_planets)
    big = torch.empty((lim + 2, stride), dtype=torch.float64, device="cuda")
    with pytest.raises(gl.GlisseError) as ex:
        S.planet_log_static(lim + 1, big)                # one step beyond the scratch
    assert ex.value.status == gl.ELIMIT and "capacity" in str(ex.value)
    S.planet_log_static(lim, big)                        # the limit itself is served ...
    want = S.planet_log(lim)
    assert np.array_equal(big[:lim + 1].cpu().numpy(), want)
    with pytest.raises(gl.GlisseError) as ex:            # ... a host buffer is not (the kernel writes it directly)
        S.planet_log_static(10, np.empty((11, stride)))
    assert ex.value.status == gl.EINVAL
    with pytest.raises(gl.GlisseError):
        S.planet_log_static(-1, big)
    S.advance(20)                                        # refusals leave the simulation usable
    S.close()
