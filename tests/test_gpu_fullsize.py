"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (C3: one ordered
subset = 36 interleaved views per launch; C2: all 360 views in one launch), on SAMPLED outputs the fp64
oracle computes one by one: seeded random rays for Ax, seeded random voxels (all views of the launch) for
A^T b.  Inputs are seeded uniform-random volumes / projections (no smoothness for fp32 error to hide
behind).  Tolerances are north_star's: 1e-5 Siddon and matched, 1e-4 interpolated and FDK (rel-L2 over the
sample).
"""
import numpy as np
import pytest

from oracle import oracle as orc
from tests import helpers as H
from workloads import make_config, phantom_for

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

N_RAYS, N_VOX = 200_000, 20_000


@pytest.fixture(scope="module")
def tg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2412_10129_b200 as m
    m.version()
    return m


def subset_geometry(name, view_ids):
    geo, ang, rec = make_config(name)
    view_ids = np.asarray(view_ids)
    if geo.rotDetector_a is not None:
        geo.rotDetector_a = geo.rotDetector_a[view_ids]
    return geo, ang[view_ids], rec


def random_volume(geo, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    v = torch.rand(geo.vol_shape, generator=g, device="cuda", dtype=torch.float32)
    return v, v.cpu().numpy()


def random_projections(geo, nA, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    p = torch.rand((nA,) + geo.proj_shape, generator=g, device="cuda", dtype=torch.float32)
    return p, p.cpu().numpy()


def check_ax(tg, geo, ang, vol_d, vol_h, mode, tol, seed):
    got = tg.Ax(vol_d, geo, ang, mode)
    ids = np.random.default_rng(seed).integers(0, got.numel(), N_RAYS)
    ref = orc.ax(vol_h, geo, ang, orc.SIDDON if mode == "siddon" else orc.INTERP, ray_ids=ids)
    g = got.reshape(-1)[torch.from_numpy(ids).cuda()].cpu().numpy().astype(np.float64)
    assert np.count_nonzero(ref) > N_RAYS // 10
    assert H.rel_l2(g, ref) <= tol
    if mode == "siddon":
        assert np.array_equal(g == 0, ref == 0)            # the same rays miss the volume


def check_atb(tg, geo, ang, proj_d, proj_h, mode, tol, seed):
    got = tg.Atb(proj_d, geo, ang, mode)
    ids = np.random.default_rng(seed).integers(0, got.numel(), N_VOX)
    ref = orc.atb(proj_h, geo, ang, orc.MATCHED if mode == "matched" else orc.FDK, vox_ids=ids)
    g = got.reshape(-1)[torch.from_numpy(ids).cuda()].cpu().numpy().astype(np.float64)
    assert H.rel_l2(g, ref) <= tol


def test_c3_full_size_siddon_and_matched(tg):
    # 512^3, 1024x768 half-fan detector; ordered subset 3 of 20 = views 3, 23, 43, ... (36 views per launch)
    geo, ang, _ = subset_geometry("C3", np.arange(3, 720, 20))
    vol_d, vol_h = random_volume(geo, 101)
    check_ax(tg, geo, ang, vol_d, vol_h, "siddon", 1e-5, 1)
    del vol_d
    proj_d, proj_h = random_projections(geo, len(ang), 102)
    for path in (0, 1):                                     # TMA-staged kernel (bench default) and gather kernel
        tg.set_atb_path(path)
        try:
            check_atb(tg, geo, ang, proj_d, proj_h, "matched", 1e-5, 2)
        finally:
            tg.set_atb_path(0)


def test_c3_full_size_weights_sampled(tg):
    # row weights 1/(A 1) of one subset at sampled rays; column weights 1/(A^T 1) at sampled voxels (P13)
    geo, ang, _ = subset_geometry("C3", np.arange(0, 720, 20))
    W = tg.row_weights(geo, ang, "siddon")
    ids = np.random.default_rng(3).integers(0, W.numel(), N_RAYS)
    a1 = orc.ax(np.ones(geo.vol_shape, np.float32), geo, ang, orc.SIDDON, ray_ids=ids)
    eps = 1e-2 * min(geo.dVoxel)
    w_ref = np.where(a1 > eps, 1.0 / np.maximum(a1, 1e-300), 0.0)
    w = W.reshape(-1)[torch.from_numpy(ids).cuda()].cpu().numpy().astype(np.float64)
    safe = np.abs(a1 - eps) > 1e-3 * eps                    # hard threshold: skip knife-edge rays
    assert np.array_equal((w == 0)[safe], (w_ref == 0)[safe])
    nz = safe & (w_ref != 0)
    assert H.rel_l2(1.0 / w[nz], 1.0 / w_ref[nz]) <= 1e-5
    V = tg.col_weights(geo, ang, "matched")
    vid = np.random.default_rng(4).integers(0, V.numel(), N_VOX)
    at1 = orc.atb(None, geo, ang, orc.MATCHED, vox_ids=vid)
    v = V.reshape(-1)[torch.from_numpy(vid).cuda()].cpu().numpy().astype(np.float64)
    assert np.all(v[at1 > 0] > 0) and H.rel_l2(1.0 / v[at1 > 0], at1[at1 > 0]) <= 1e-5


def test_c2_full_size_interp_and_fdk(tg):
    # 256^3, 512x512 detector: interpolated Ax on 36 of the 360 views, FDK-weighted A^T b over all 360 views
    geo, ang, _ = subset_geometry("C2", np.arange(0, 360, 10))
    vol_d, vol_h = random_volume(geo, 201)
    check_ax(tg, geo, ang, vol_d, vol_h, "interp", 1e-4, 5)
    geo, ang, _ = subset_geometry("C2", np.arange(360))
    proj_d, proj_h = random_projections(geo, 360, 202)
    check_atb(tg, geo, ang, proj_d, proj_h, "fdk", 1e-4, 6)


def test_c4_full_size_tilted_detectors(tg):
    # 1024^3 (4.3 GB), 1536^2 detector, per-view detector roll/pitch/yaw and COR offset: interpolated Ax on 4
    # views, matched A^T b on 16 views (the general, non z-aligned inner loop of the TMA kernel)
    geo, ang, _ = subset_geometry("C4", np.arange(0, 1600, 400))
    vol_d, vol_h = random_volume(geo, 301)
    check_ax(tg, geo, ang, vol_d, vol_h, "interp", 1e-4, 7)
    del vol_d, vol_h
    torch.cuda.empty_cache()
    geo, ang, _ = subset_geometry("C4", np.arange(0, 1600, 100))
    proj_d, proj_h = random_projections(geo, len(ang), 302)
    check_atb(tg, geo, ang, proj_d, proj_h, "matched", 1e-5, 8)


def test_c3_full_size_ossart_teacher_forced(tg):
    """north_star's target run, 20 iterations x 20 ordered subsets of OS-SART on the full C3 problem (its phantom, Poisson noise on
    I0 = 1e5, half-fan detector) through the plan bench.py times, checked against the oracle by teacher forcing (SURVEY.md section
    8(d)): before subset 0 of iteration 1, subset 7 of iteration 10 and subset 19 of iteration 20 the GPU's iterate is handed to
    the oracle, which applies ONE ordered-subset update of reading P13 / PAPER.md:115 to 20 000 sampled voxels,
    x_j <- max(0, x_j + V_j (A_s^T W (b_s - A_s x))_j); the GPU takes the same step through THE 20-SUBSET PLAN ITSELF
    (tigre_plan_ossart_subsets: its own W_s, V_s, view lists and offsets).  The oracle evaluates A_s x and A_s 1 only at the
    detector pixels the sampled voxels' bilinear taps touch (their indices come from the oracle's own voxel map)."""
    geo, ang, rec = make_config("C3")
    nA, (nu, nv) = len(ang), geo.nDetector
    subsets = [np.arange(s, nA, 20) for s in range(20)]
    vol_h = phantom_for(rec, geo)
    b_d = tg.Ax(torch.from_numpy(vol_h).cuda(), geo, ang, "siddon")
    gen = torch.Generator(device="cuda").manual_seed(rec["seed"])
    b_d = -torch.log(torch.clamp(torch.poisson(1e5 * torch.exp(-b_d), generator=gen), min=1.0) / 1e5)    # reading P18, drawn once
    b_h = b_d.cpu().numpy()
    del vol_h
    n_vox = 20000
    ids = np.random.default_rng(402).integers(0, int(np.prod(geo.vol_shape)), n_vox)
    ids_d = torch.from_numpy(ids).cuda()
    eps_w = 1e-2 * min(geo.dVoxel)
    ones = np.ones(geo.vol_shape, np.float32)

    plan = tg.OssartPlan(geo, ang, subsets, "siddon", "matched")
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    done = 0                                                           # full iterations applied to x
    try:
        for it, s in ((1, 0), (10, 7), (20, 19)):
            if it - 1 > done:
                plan.iterate(b_d, x, it - 1 - done, want_resid=False)
                done = it - 1
            plan.iterate_subsets(b_d, x, 0, s)                          # subsets 0 .. s-1 of iteration `it`
            x_prev = x.cpu().numpy()
            plan.iterate_subsets(b_d, x, s, s + 1)                      # the step under test
            got = x.reshape(-1)[ids_d].cpu().numpy().astype(np.float64)
            plan.iterate_subsets(b_d, x, s + 1, len(subsets))           # finish the iteration
            done = it
            # ---- the oracle's update of the sampled voxels with subset s
            geo_s, ang_s, _ = subset_geometry("C3", subsets[s])
            nS = len(subsets[s])
            b_s = b_h[subsets[s]].astype(np.float64)
            at1, fuv = orc.atb(None, geo_s, ang_s, orc.MATCHED, vox_ids=ids, return_fuv=True)
            iu0, iv0 = np.floor(fuv[..., 0]).astype(np.int64), np.floor(fuv[..., 1]).astype(np.int64)     # [n_vox][nS]
            ia = np.broadcast_to(np.arange(nS)[None, :], iu0.shape)
            rays = []
            for du in (0, 1):
                for dv in (0, 1):
                    u, v = iu0 + du, iv0 + dv
                    ok = (u >= 0) & (u < nu) & (v >= 0) & (v < nv)
                    rays.append(((ia * nv + v) * nu + u)[ok])
            rid = np.unique(np.concatenate(rays))
            a1 = orc.ax(ones, geo_s, ang_s, orc.SIDDON, ray_ids=rid)
            W = np.where(a1 > eps_w, 1.0 / np.maximum(a1, 1e-300), 0.0)
            seen = at1 > 1e-4 * at1.max()          # V's own threshold is 1e-6 max_j (A^T 1)_j over the volume: stay clear of it
            assert np.count_nonzero(seen) > n_vox // 2
            V = np.where(seen, 1.0 / np.maximum(at1, 1e-300), 0.0)
            r = np.zeros(nS * nv * nu)
            r[rid] = W * (b_s.reshape(-1)[rid] - orc.ax(x_prev, geo_s, ang_s, orc.SIDDON, ray_ids=rid))
            g = orc.atb(r.reshape(nS, nv, nu), geo_s, ang_s, orc.MATCHED, vox_ids=ids)
            xp = x_prev.reshape(-1)[ids].astype(np.float64)
            ref = np.maximum(xp + V * g, 0.0)
            assert H.rel_l2(got[seen], ref[seen]) <= 1e-5, (it, s)
            moved = seen & ((ref > 0) | (got > 0))
            assert H.rel_l2((got - xp)[moved], (ref - xp)[moved]) <= 1e-4, (it, s)      # the update itself
            assert np.isfinite(got).all()
    finally:
        plan.close()


def test_c4_full_size_cgls_two_iterations_teacher_forced(tg):
    """configs[3]: CGLS on the full C4 problem (1024^3, 1600 views of 1536^2, per-view detector roll / pitch / yaw, COR offset;
    interpolated Ax, matched A^T b) through tigre_cgls, first two iterations, against the textbook recurrences (DESIGN.md O-F)
    with the oracle's operators on 5000 sampled voxels.  The global scalars (gamma, ||A p||^2) are formed in fp64 from arrays
    the SAME library calls produce outside the driver (teacher forcing: the oracle cannot form a 3.8e9-ray norm), so this
    checks (i) the operators at full size inside the driver, (ii) the recurrences, (iii) the residual history.
    Tolerance: x_1 = alpha_0 A^T b is linear in one matched backprojection (1e-5) times a ratio of two norms that carry the
    interpolated projector's 1e-4: 3e-4; iteration 2 adds a second projection / backprojection pair: 6e-4."""
    if torch.cuda.mem_get_info()[0] < 90e9:
        pytest.skip("needs 90 GB of free HBM")
    geo, ang, rec = make_config("C4")
    nA = len(ang)
    gen = torch.Generator(device="cuda").manual_seed(rec["seed"])
    vol = torch.rand(geo.vol_shape, generator=gen, device="cuda") * 0.02
    b = tg.Ax(vol, geo, ang, "interp")
    del vol
    ids = np.random.default_rng(77).integers(0, int(np.prod(geo.vol_shape)), 5000)
    ids_d = torch.from_numpy(ids).cuda()

    def dot(a, c):
        return float((a.double().reshape(-1) * c.double().reshape(-1)).sum()) if a.numel() < 2 ** 31 else \
            sum(float((a[i].double() * c[i].double()).sum()) for i in range(a.shape[0]))

    x2, hist = tg.cgls(b, geo, ang, 2, "interp", "matched")
    x1, _ = tg.cgls(b, geo, ang, 1, "interp", "matched")
    got1 = x1.reshape(-1)[ids_d].cpu().numpy().astype(np.float64)
    got2 = x2.reshape(-1)[ids_d].cpu().numpy().astype(np.float64)
    del x1, x2
    # ---- iteration 1: s0 = A^T b, p0 = s0, q0 = A p0, alpha0 = |s0|^2 / |q0|^2, x1 = alpha0 p0, r1 = b - alpha0 q0
    s0 = tg.Atb(b, geo, ang, "matched")
    q0 = tg.Ax(s0, geo, ang, "interp")
    gamma0, qq0 = dot(s0, s0), dot(q0, q0)
    alpha0 = gamma0 / qq0
    b_h = b.cpu().numpy()
    s0_ref = orc.atb(b_h, geo, ang, orc.MATCHED, vox_ids=ids)
    assert H.rel_l2(got1, alpha0 * s0_ref) <= 3e-4
    r1 = b - float(alpha0) * q0
    assert hist[0] == pytest.approx(np.sqrt(dot(r1, r1)), rel=1e-4)
    del q0, b, b_h
    # ---- iteration 2: s1 = A^T r1, beta = |s1|^2 / gamma0, p1 = s1 + beta p0, alpha1 = |s1|^2 / |A p1|^2, x2 = x1 + alpha1 p1
    s1 = tg.Atb(r1, geo, ang, "matched")
    gamma1 = dot(s1, s1)
    beta = gamma1 / gamma0
    p1 = s1 + float(beta) * s0
    del s1
    q1 = tg.Ax(p1, geo, ang, "interp")
    alpha1 = gamma1 / dot(q1, q1)
    r1_h = r1.cpu().numpy()
    del r1, q1, p1, s0
    s1_ref = orc.atb(r1_h, geo, ang, orc.MATCHED, vox_ids=ids)
    ref2 = alpha0 * s0_ref + alpha1 * (s1_ref + beta * s0_ref)
    assert H.rel_l2(got2, ref2) <= 6e-4
    assert H.rel_l2(got2 - got1, alpha1 * (s1_ref + beta * s0_ref)) <= 2e-3          # the second step on its own
