"""pm_objective_noalloc (include/pm.h): the mesh objective as an entry point that allocates nothing (static device scratch),
checked against the existing path -- pm_set_state + pm_objective + pm_get_objective of a ctx -- on two calls in a row.

Collected last on purpose (pytest -x stops at the first failure).  Passes alone in a fresh process and
after the other tests: it needs nothing but its own inputs."""
import numpy as np
import pytest

from paper_2211_09815_b200 import inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pmlib():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_2211_09815_b200 import binding
    return binding


def test_objective_noalloc_matches_the_ctx_path_on_two_calls(pmlib):
    mesh, lattice, omm = (64, 48, 40), (32, 24, 20), 0.3          # 122880 mesh points: two scratch blocks, ragged second one
    a = inputs.a_schedule(0.25, 2)
    nbar = np.prod(lattice) / np.prod(mesh)
    pm = pmlib.PM(mesh, lattice, omm, a)
    J = torch.zeros(1, dtype=torch.float64, device="cuda")
    resid = torch.empty(mesh, dtype=torch.float32, device="cuda")
    q = np.stack(np.meshgrid(*[np.arange(lattice[d], dtype=np.float32) * 2 for d in range(3)], indexing="ij"), axis=-1).reshape(-1, 3)
    for call, seed in enumerate((1, 5)):                           # two calls in a row: the scratch keeps the first one's contents
        s = inputs.zeldovich_displacement(lattice, mesh, seed=seed, rms=0.8 + call)
        s = (np.round(s * 65536.0) / 65536.0).astype(np.float32)   # q + s exact in fp32: both paths see the same positions
        target = inputs.lognormal_target(mesh, seed=seed + 1, sigma=0.7)
        sd, td = torch.from_numpy(s).cuda(), torch.from_numpy(target).cuda()
        # existing path: the ctx's objective on the state (q + s)
        pm.set_state(sd, torch.zeros_like(sd))
        pm.objective(td)
        J_ctx = pm.get_objective()
        # new entry point on the density of the same positions (existing pm_scatter), nothing allocated by libpm
        rho = pm.scatter(torch.from_numpy(q + s).cuda())
        mem0 = torch.cuda.memory_allocated()
        pmlib.objective_noalloc(rho, td, nbar, J, resid=resid)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == mem0
        assert J_ctx > 0 and abs(float(J[0]) - J_ctx) <= 1e-6 * J_ctx, (float(J[0]), J_ctx)
        r = rho.double() / nbar - 1.0 - td.double()
        assert abs(float(J[0]) - 0.5 * float((r * r).sum())) <= 1e-6 * J_ctx
        assert float((resid.double() - r).abs().max()) <= 1e-5 * float(r.abs().max())
    pm.close()


def test_objective_noalloc_rejects_sizes_beyond_the_maximum(pmlib):
    x = torch.zeros(16, dtype=torch.float32, device="cuda")
    J = torch.zeros(1, dtype=torch.float64, device="cuda")
    rc = pmlib._lib.pm_objective_noalloc(pmlib.PM_NOALLOC_MAX_N + 1, x.data_ptr(), x.data_ptr(), 1.0, None, J.data_ptr(), None)
    assert rc == pmlib.PM_EINVAL
    assert b"PM_NOALLOC_MAX_N" in pmlib._lib.pm_last_error(None)
    assert pmlib._lib.pm_noalloc_setup() == pmlib.PM_OK
