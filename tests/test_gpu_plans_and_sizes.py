"""GPU parity on the code paths only the larger configs take (run on the B200 box with `-m gpu`):

  * every radix plan of the library's own FFT passes (axes of 16 ... 1024 points) against the ORACLE's force and
    force VJP on thin meshes the oracle finishes in seconds;
  * the whole forward + adjoint run of configs[0] with CIC deconvolution switched on (reading R12);
  * the two-stream adjoint step on a clustered state (heavy tiles: split scatter tiles, gather chunks in the work
    queues of both streams at once), bit-identical to the one-stream order, under a host-side timeout;
  * configs[3]/configs[4] sizes (512^3 particles, 1024^3 mesh): pm_scatter against the oracle's scatter on the whole
    mesh (unit mass) and on sub-boxes (3 components), gathers on sampled particles, for the real configs[4] inputs;
    own-FFT path against the cuFFT path for pm_force / pm_force_vjp at 1024^3.
"""
import gc

import numpy as np
import pytest

from paper_2211_09815_b200 import inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.sqrt(np.sum((a - b) ** 2) / max(np.sum(b ** 2), 1e-300)))


@pytest.fixture(scope="module")
def pmlib():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_2211_09815_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


# One mesh per plan: x / y axes of 16 (radix 16), 32 (8 x 4), 64 (16 x 4), 128 (16 x 8), 256 (16 x 16), 512 (8 x 16 x 4),
# 1024 (16 x 16 x 4); z axes whose half length Nz/2 runs through 8 ... 512.  Thin in the other directions.
PLAN_MESHES = [
    (512, 16, 32), (16, 512, 32), (32, 16, 512), (16, 32, 1024), (32, 32, 32), (1024, 16, 16), (16, 1024, 16),
    (128, 64, 16), (64, 128, 256), (256, 16, 64), (16, 256, 128),
]


# deconvolution is covered on three of the plans (a 512, a 1024 x axis and a 1024 z axis)
PLAN_CASES = [(m, 0) for m in PLAN_MESHES] + [((512, 16, 32), 1), ((16, 32, 1024), 1), ((1024, 16, 16), 1)]


@pytest.mark.parametrize("mesh,deconv", PLAN_CASES)
def test_own_fft_plans_against_oracle(pmlib, orc, mesh, deconv, monkeypatch):
    """pm_force / pm_force_vjp through the own z, y and fused x passes against the oracle (eq. 11 L127-131 and its
    transpose), rel L2 <= 1e-5, on a mesh with one long axis per radix plan."""
    monkeypatch.setenv("PM_FFT", "own")   # also above the default own-FFT size limit, if any
    lattice = tuple(n // 2 for n in mesh)
    rng = np.random.default_rng(41)
    pm = pmlib.PM(mesh, lattice, 0.3, [0.5, 1.0], deconvolve=deconv)
    assert pm.np == int(np.prod(lattice))
    s = rng.normal(0, 1.2, (pm.np, 3))
    x = orc.positions(mesh, lattice, s).astype(np.float32)
    pi = rng.standard_normal((pm.np, 3)).astype(np.float32)
    acc, alpha = pm.force_vjp(dev(x), dev(pi))
    own, fft = pm.launch_count()
    assert fft == 0, "the own FFT path must not call cuFFT"
    acc_o = orc.force(mesh, 0.3, x, deconv=deconv)
    alpha_o = orc.force_vjp(mesh, 0.3, x, pi, deconv=deconv)
    assert rel_l2(acc.cpu().numpy(), acc_o) <= 1e-5
    assert rel_l2(alpha.cpu().numpy(), alpha_o) <= 1e-5
    pm.close()


def _cfg0_inputs(orc, deconv):
    cfg = inputs.config(0)
    s0 = inputs.zeldovich_displacement(cfg["lattice"], cfg["mesh"], seed=1, rms=0.3)
    ratio = orc.p_over_s(cfg["omega_m"], cfg["a"][0])
    p0 = (s0.astype(np.float64) * ratio).astype(np.float32)
    s0t = inputs.zeldovich_displacement(cfg["lattice"], cfg["mesh"], seed=2, rms=0.3)
    p0t = (s0t.astype(np.float64) * ratio).astype(np.float32)
    s_nt, _, _ = orc.run_fwd(cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"], s0t, p0t, deconv=deconv)
    xt = orc.positions(cfg["mesh"], cfg["lattice"], s_nt)
    nbar = np.prod(cfg["lattice"]) / np.prod(cfg["mesh"])
    target = (orc.scatter(cfg["mesh"], xt) / nbar - 1.0).astype(np.float32)
    return cfg, s0, p0, target


@pytest.mark.parametrize("fft", ["own", "cufft"])
def test_config0_whole_run_with_deconvolution(pmlib, orc, fft, monkeypatch):
    """SURVEY reading 12: whole-run parity at configs[0] in BOTH deconvolution modes (mode 0 is in test_gpu_parity.py).

    Deconvolution multiplies the force at the mesh Nyquist by up to (pi/2)^12 and makes the 16-step run ill-conditioned:
    the ORACLE's own gradient moves by 3e-2 when its input displacements are changed by 1e-7 cell (4 ulp of the fp32
    inputs).  The gradient tolerance is therefore measured, not assumed (R28): twice the change of the oracle's
    gradient under such a perturbation, and never below north_star's 1e-3 (which is what holds without deconvolution,
    where the same measurement gives 2e-4).  Positions, objective and the exact reversal keep north_star's numbers."""
    monkeypatch.setenv("PM_FFT", fft)
    cfg, s0, p0, target = _cfg0_inputs(orc, 1)
    args = (cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"])
    ref = orc.run_fwd_adj(*args, s0, p0, target, deconv=1)
    s0_pert = s0.astype(np.float64) + 1e-7 * np.random.default_rng(5).standard_normal(s0.shape)
    ref_pert = orc.run_fwd_adj(*args, s0_pert, p0, target, deconv=1)
    pm = pmlib.PM(*args, deconvolve=1)
    out = pm.run_fwd_adj(dev(s0), dev(p0), dev(target))
    s_n = out["s_n"].cpu().numpy().astype(np.float64)
    rms = np.sqrt(np.mean(np.sum((s_n - ref["s_n"]) ** 2, axis=1)))
    assert rms <= 1e-4, f"final positions rms {rms} cell"
    assert abs(out["J"] - ref["J"]) <= 1e-4 * abs(ref["J"])
    for k in ("xi0", "pi0", "dJ_ds0"):
        cond = rel_l2(ref_pert[k], ref[k])
        assert cond >= 1e-3, "the premise of this tolerance (an ill-conditioned run) no longer holds: assert 1e-3 instead"
        e = rel_l2(out[k].cpu().numpy(), ref[k])
        assert e <= 2.0 * cond, f"{k} rel L2 {e} (oracle's own change under a 1e-7-cell perturbation: {cond})"
        # the bulk of the particles is not in the chaotic regime: median per-particle error at north_star's number
        a, b = out[k].cpu().numpy().astype(np.float64), ref[k]
        med = np.median(np.sqrt(np.sum((a - b) ** 2, axis=1) / np.sum(b ** 2, axis=1)))
        assert med <= 1e-3, f"{k} median per-particle relative error {med}"
    s_q = np.rint(s0.astype(np.float64) * 2.0 ** 32) / 2.0 ** 32
    assert np.array_equal(out["s_rec"].cpu().numpy(), s_q.astype(np.float32))
    pm.close()


def _clustered_state(L, N, n_blobs):
    """displacements that put the lattice particles on the configs[4] blob distribution (generation order)"""
    mesh = (N, N, N)
    x = inputs.blob_positions(L ** 3, mesh, seed=3, n_blobs=n_blobs, order="generation").astype(np.float64)
    q = np.stack(np.meshgrid(*[np.arange(L) * (N // L)] * 3, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    s = x - q
    s -= N * np.rint(s / N)          # minimum image: |s| <= N/2
    return mesh, s.astype(np.float32)


@pytest.mark.timeout(600, method="thread")
def test_two_stream_adjoint_on_clustered_state(pmlib, monkeypatch):
    """Adjoint steps on a state with collapsed clumps: the unit-mass scatter splits heavy tiles through the work queue
    of the caller's stream while the valued scatter / gathers of the other branch run on stream2 with their own
    queue.  Must terminate (a broken queue invariant raises PMError through the watchdog instead of hanging) and
    agree bit for bit with the one-stream order."""
    L, N = 128, 256
    mesh, s0 = _clustered_state(L, N, 313)
    a = inputs.a_schedule(0.5, 3)
    rng = np.random.default_rng(9)
    p0 = (0.05 * rng.standard_normal(s0.shape)).astype(np.float32)
    xi = rng.standard_normal(s0.shape).astype(np.float32)
    pi = rng.standard_normal(s0.shape).astype(np.float32)
    outs = {}
    for mode in ("1", "0"):
        monkeypatch.setenv("PM_OVERLAP", mode)
        pm = pmlib.PM(mesh, (L,) * 3, 0.3, a)
        pm.set_state(dev(s0), dev(p0))
        for i in range(1, 4):
            pm.step_fwd(i)
        pm.set_adjoint(dev(xi), dev(pi))
        for i in range(3, 0, -1):
            pm.step_adj(i)
        torch.cuda.synchronize()
        outs[mode] = [t.clone() for t in pm.get_adjoint()] + list(pm.get_state())
        pm.get_objective()   # synchronises and checks the watchdog flags of both streams
        pm.close()
    for u, v in zip(outs["1"], outs["0"]):
        assert torch.equal(u, v)
    # reversal is exact on this state too
    s_q = np.rint(s0.astype(np.float64) * 2.0 ** 32) / 2.0 ** 32
    assert np.array_equal(outs["1"][3].cpu().numpy(), s_q.astype(np.float32))


# ---- configs[3] / configs[4] sizes ------------------------------------------------------------------------------------
BIG_L, BIG_N = 512, 1024


def test_config3_force_vjp_own_fft_vs_cufft(pmlib, monkeypatch):
    """pm_force / pm_force_vjp at 1024^3 on the configs[3] initial state: the library's own fp32 transform passes and the
    cuFFT fp32 + stand-alone k-space kernel path, each against the fp64-transform mode (PM_FLAG_FP64_TRANSFORMS: cuFFT
    D2Z / Z2D and fp64 k-space kernels; three implementations of eq. 11 and its transpose, each compared with the oracle
    on the smaller meshes above).  The oracle itself needs ~70 GB of host memory for one force at 1024^3 (DESIGN.md
    section 7), so at this size the paths check each other.  Tolerance: on the INITIAL state the mesh rms is dominated by
    the (force-free) pattern of the barely displaced particle lattice, so the fp32 transforms' rounding (3e-7 of the mesh
    rms at 30 butterfly levels) is 2e-6 of the small physical force (measured: own vs cuFFT 2.9e-6); 5e-6 asserted."""
    cfg = inputs.config(3)
    s0 = inputs.zeldovich_displacement(cfg["lattice"], cfg["mesh"], seed=1, rms=0.3)
    q = np.stack(np.meshgrid(*[np.arange(BIG_L, dtype=np.float32) * 2] * 3, indexing="ij"), axis=-1).reshape(-1, 3)
    x = q + s0
    rng = np.random.default_rng(29)
    pi = rng.standard_normal(x.shape).astype(np.float32)
    res = {}
    for mode in ("own", "cufft", "fp64"):
        monkeypatch.setenv("PM_FFT", "cufft" if mode == "fp64" else mode)
        pm = pmlib.PM(cfg["mesh"], cfg["lattice"], cfg["omega_m"], [1.0],
                      flags=pmlib.PM_FLAG_FP64_TRANSFORMS if mode == "fp64" else 0)
        acc, alpha = pm.force_vjp(torch.from_numpy(x).cuda(), torch.from_numpy(pi).cuda())
        own, fft = pm.launch_count()
        assert (fft == 0) == (mode == "own")
        res[mode] = (acc.cpu().numpy(), alpha.cpu().numpy())
        pm.close()
        del acc, alpha
        torch.cuda.empty_cache()
    for mode in ("own", "cufft"):
        assert rel_l2(res[mode][0], res["fp64"][0]) <= 5e-6, mode
        assert rel_l2(res[mode][1], res["fp64"][1]) <= 5e-6, mode
    tot = np.abs(res["own"][0].astype(np.float64).sum(axis=0))
    assert np.all(tot <= 1e-5 * np.abs(res["own"][0]).sum(axis=0))      # P3 momentum conservation at full size


def test_config3_whole_run_exact_reversal_and_fp64_transform_cross_check(pmlib):
    """configs[3] (512^3 particles, 1024^3 mesh, 100 KDK steps) end to end.  The oracle cannot run this size on the box
    (hours, ~70 GB per force), so what is checked is what holds at any size: (1) the reverse pass returns the quantised
    initial state BIT FOR BIT at full size (134 M particles, 100 steps forward and back, own 1024-point transform passes);
    (2) the fp32 path against the fp64-transform mode of the same library (the mode that sits within 1.7e-6 cell and 1.5e-4
    of the oracle at configs[1]): final positions within north_star's 1e-4 cell rms, objective 1e-4,
    median per-particle gradient difference 1e-3 on 65536 sampled particles.  A stand-in for the oracle, stated as such."""
    gc.collect()
    torch.cuda.empty_cache()            # blocks cached by the earlier tests of this process count as used otherwise
    free, _ = torch.cuda.mem_get_info()
    cfg = inputs.config(3)
    need = pmlib.workspace_bytes(cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"], flags=pmlib.PM_FLAG_FP64_TRANSFORMS)
    if free < need + (24 << 30):
        pytest.fail(f"configs[3] in the fp64-transform mode needs {need / 2**30:.0f} GiB of workspace; {free / 2**30:.0f} GiB free")
    s0 = inputs.zeldovich_displacement(cfg["lattice"], cfg["mesh"], seed=1, rms=0.3)
    g = pmlib.host_growth(cfg["omega_m"], cfg["a"][0])
    p0 = (s0.astype(np.float64) * (g[2] / g[0])).astype(np.float32)
    target = inputs.lognormal_target(cfg["mesh"], seed=2, sigma=1.0)
    dv = [torch.from_numpy(v).cuda() for v in (s0, p0, target)]
    del target
    idx = np.sort(np.random.default_rng(7).choice(s0.shape[0], size=65536, replace=False))
    res = {}
    for mode, flags in (("fp32", 0), ("fp64t", pmlib.PM_FLAG_FP64_TRANSFORMS)):
        pm = pmlib.PM(cfg["mesh"], cfg["lattice"], cfg["omega_m"], cfg["a"], flags=flags)
        out = pm.run_fwd_adj(*dv)
        own, fft = pm.launch_count()
        assert (fft == 0) == (mode == "fp32")             # the fp32 path runs its own transform passes at 1024^3
        s_q = np.rint(s0.astype(np.float64) * 2.0 ** 32) / 2.0 ** 32
        assert np.array_equal(out["s_rec"].cpu().numpy(), s_q.astype(np.float32)), f"{mode}: reverse integration is not exact"
        res[mode] = {k: out[k].cpu().numpy()[idx].astype(np.float64) for k in ("s_n", "dJ_ds0")}
        res[mode]["J"] = out["J"]
        pm.close()
        del out, pm
        torch.cuda.empty_cache()
    rms = float(np.sqrt(np.mean(np.sum((res["fp32"]["s_n"] - res["fp64t"]["s_n"]) ** 2, axis=1))))
    a, b = res["fp32"]["dJ_ds0"], res["fp64t"]["dJ_ds0"]
    e2, n2 = np.sum((a - b) ** 2, axis=1), np.sum(b ** 2, axis=1)
    print(f"configs[3] fp32 vs fp64-transform mode: positions rms {rms:.3e} cell, J rel {abs(res['fp32']['J'] / res['fp64t']['J'] - 1):.2e}, "
          f"dJ/ds0 rel L2 {np.sqrt(e2.sum() / n2.sum()):.3e}, median {np.median(np.sqrt(e2 / n2)):.3e}")
    assert rms <= 1e-4
    assert abs(res["fp32"]["J"] / res["fp64t"]["J"] - 1) <= 1e-4
    assert np.median(np.sqrt(e2 / n2)) <= 1e-3


@pytest.fixture(scope="module")
def big(pmlib):
    """One ctx of the configs[3] geometry (69.5 GB workspace) shared by the full-size kernel tests."""
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    need = pmlib.workspace_bytes((BIG_N,) * 3, (BIG_L,) * 3, 0.3, [1.0])
    if free < need + (24 << 30):
        pytest.fail(f"configs[3] needs {need / 2**30:.0f} GiB of workspace; {free / 2**30:.0f} GiB free on this device")
    pm = pmlib.PM((BIG_N,) * 3, (BIG_L,) * 3, 0.3, [1.0])
    yield pm
    pm.close()


def _subbox_scatter(orc, x, val, lo, size):
    """The oracle's scatter restricted to the mesh points [lo, lo + size)^3 of the periodic 1024^3 mesh: every particle
    within one cell of the box is deposited (serially, eq. 10) on a private periodic mesh of 2 x size points, shifted so
    that the box sits in its middle; deposits from outside the box never reach its interior."""
    N = BIG_N
    d = np.mod(x.astype(np.float64) - (np.asarray(lo, dtype=np.float64) - 1.0), N)     # distance above lo - 1
    sel = np.all(d < size + 2.0, axis=1)
    m = 2 * size
    xs = d[sel] - 1.0 + size // 2                                                       # box starts at size // 2
    out = orc.scatter((m, m, m), xs, None if val is None else val[sel])
    h = size // 2
    return out[..., h:h + size, h:h + size, h:h + size], int(sel.sum())


def test_config4_inputs_full_size_kernel_parity(pmlib, orc, big):
    """The real configs[4] inputs (512^3 particles, 20000 blobs, 1024^3 mesh).  Generation order: pm_scatter (unit mass)
    against the oracle's serial scatter on the WHOLE mesh; the 3-component scatter on sub-boxes around the densest
    cells and at the periodic corner; gathers and weight-gradient gathers on 20000 sampled particles.  Random memory
    order (the same particles permuted): every result must equal the generation-order one BIT FOR BIT -- the meshes
    because the scatters accumulate in integers, the per-particle outputs because they depend on the particle alone --
    which carries the oracle comparison over without a second 134 M-particle serial scatter on the host.  This exercises
    the 64-bit index paths, the 1024-axis tile counts and the work queues / accumulator pool at their real load."""
    pm = big
    mesh = (BIG_N,) * 3
    npart = BIG_L ** 3
    x = inputs.blob_positions(npart, mesh, seed=3, n_blobs=20000, order="generation")
    xd = torch.from_numpy(x).cuda()
    rng = np.random.default_rng(23)
    # --- unit-mass scatter, whole mesh, compared slab by slab (the fp64 mesh of the oracle is 8.6 GB)
    rho_d = pm.scatter(xd)
    rho = rho_d.cpu().numpy()
    rho_o = orc.scatter(mesh, x)
    assert rho_o.max() > 100.0
    num = den = tot = 0.0
    for i in range(0, BIG_N, 64):
        a = rho[i:i + 64].astype(np.float64)
        b = rho_o[i:i + 64]
        num += float(np.sum((a - b) ** 2))
        den += float(np.sum(b ** 2))
        tot += float(a.sum())
    assert np.sqrt(num / den) <= 1e-5
    assert abs(tot - npart) <= 1e-6 * npart
    # densest cells (for the sub-boxes of the valued scatter) before the big arrays go
    flat = np.argpartition(rho_o.reshape(-1), -4)[-4:]
    peaks = [np.unravel_index(int(f), mesh) for f in flat]
    del rho, rho_o
    # --- 3-component scatter on sub-boxes of 32^3 points: two around the densest cells, the periodic corner, one random
    val = (rng.standard_normal((npart, 3)) * np.exp(rng.normal(0, 1.5, (npart, 1)))).astype(np.float32)
    vd = torch.from_numpy(val).cuda()
    m3 = pm.scatter(xd, vd)
    assert abs(float(m3.double().sum()) - float(val.astype(np.float64).sum())) <= 1e-6 * float(np.abs(val).sum())
    boxes = [tuple((int(p[d]) - 16) % BIG_N for d in range(3)) for p in peaks[:2]] + [(BIG_N - 16,) * 3, (300, 700, 100)]
    for lo in boxes:
        ref, nsel = _subbox_scatter(orc, x, val, lo, 32)
        ix = [torch.from_numpy((np.arange(32) + lo[d]) % BIG_N).cuda() for d in range(3)]
        got = m3[:, ix[0]][:, :, ix[1]][:, :, :, ix[2]].cpu().numpy()
        assert nsel > 0 and rel_l2(got, ref) <= 1e-5, f"box {lo}"
    del val
    # --- the same particles in random memory order: bit-identical meshes
    perm = torch.from_numpy(np.random.default_rng(29).permutation(npart)).cuda()
    xr = xd[perm].contiguous()
    assert torch.equal(pm.scatter(xr), rho_d), "unit-mass scatter depends on the memory order"
    del rho_d
    vr = vd[perm].contiguous()
    del vd
    m3r = pm.scatter(xr, vr)
    assert torch.equal(m3r, m3), "valued scatter depends on the memory order"
    del m3, m3r, vr
    torch.cuda.empty_cache()
    # --- gathers on sampled particles (generation order against the oracle, random order against generation order)
    gen = torch.Generator(device="cuda").manual_seed(5)
    fd = torch.randn((3,) + mesh, device="cuda", generator=gen)
    idx = np.sort(rng.choice(npart, 20000, replace=False))
    g3d = pm.gather(xd, fd)
    g3 = g3d[torch.from_numpy(idx).cuda()].cpu().numpy()
    f = fd.cpu().numpy()
    assert rel_l2(g3, orc.gather(mesh, x[idx], f)) <= 1e-5
    assert torch.equal(pm.gather(xr, fd), g3d[perm]), "gather depends on the memory order"
    del g3d
    cot = rng.standard_normal((npart, 3)).astype(np.float32)
    cd = torch.from_numpy(cot).cuda()
    ggd = pm.gather_grad(xd, fd, cd)
    gg = ggd[torch.from_numpy(idx).cuda()].cpu().numpy()
    assert rel_l2(gg, orc.gather_grad(mesh, x[idx], f, cot[idx])) <= 1e-5
    assert torch.equal(pm.gather_grad(xr, fd, cd[perm].contiguous()), ggd[perm]), "weight-gradient gather depends on the memory order"
    del ggd, cd
    gs = pm.gather_grad(xd, fd[0].contiguous())[torch.from_numpy(idx).cuda()].cpu().numpy()
    assert rel_l2(gs, orc.gather_grad(mesh, x[idx], f[0])) <= 1e-5
    pm.get_objective()   # synchronises and checks the work-queue watchdog
