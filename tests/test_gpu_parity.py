"""GPU-vs-oracle parity of the hot path (run on the B200 box: pytest -m gpu).

Every test calls the CUDA path through the C ABI (via the same-name Python binding) and compares it
with the fp64 oracle on the same seeded inputs.  Tolerances are the ones BASELINE.json's north_star
states: each amplitude within 1e-5 * sum_j |w_j| of the oracle, each cross section within relative
1e-3 wherever it exceeds 1e-6 of its maximum.
"""
import numpy as np
import pytest

import nms_inputs as ni
from nms_inputs import KIND_INDEX as KI

pytestmark = pytest.mark.gpu

AMP_TOL = 1e-5      # x sum_j |w_cj|
XS_RTOL = 1e-3      # relative, where |oracle| > XS_FLOOR * max|oracle|
XS_FLOOR = 1e-6


@pytest.fixture(scope="module")
def nms():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2601_18444_b200 as mod
    return mod


@pytest.fixture()
def ctx(nms):
    c = nms.Context(0)
    yield c.h
    c.close()


def _t(a, dtype=None):
    import torch
    if a is None:
        return None
    return torch.as_tensor(np.ascontiguousarray(a), device="cuda") if dtype is None else torch.as_tensor(np.ascontiguousarray(a, dtype=dtype), device="cuda")


def _upload(nms, h, wl, R=None):
    pos, N, m = _t(wl.pos), _t(wl.N), _t(wl.m)
    nms.nms_set_sample(h, pos, N, m, wl.R if R is None else R)
    if wl.offsets is not None:
        nms.nms_set_particles(h, wl.offsets, _t(wl.centres))
    nms.nms_set_polarization(h, wl.P)
    return pos, N, m


def assert_amplitudes(A_gpu, A_ref, wsum, label=""):
    """|A_gpu - A_ref| <= 1e-5 sum|w_c| per component; exactly zero where the component has no weight."""
    for c in range(4):
        for part in (0, 1):
            d = np.abs(A_gpu[2 * c + part].astype(np.float64) - A_ref[2 * c + part])
            if wsum[c] == 0.0:
                assert np.all(A_gpu[2 * c + part] == 0.0), f"{label}: component {c} must be exactly zero"
            else:
                worst = d.max() / wsum[c]
                assert worst <= AMP_TOL, f"{label}: amplitude plane {2 * c + part}: max err {worst:.3e} x sum|w|"


NULL_LEVEL = 1e-9   # a signed map below this fraction of its parent's maximum is "null by symmetry"
SIGNED = (KI["NM"], KI["CHI"])


def parent_maps(oracle_mod, A, th, P=None, sN=1.0, sM=1.0, invV=1.0):
    """Parent half-sum channels of the two signed difference channels (reading 16):
    NM = (PP - MM)/2 with parent (PP + MM)/2 = NUC + PROJ (Eq. 16-17); CHI = (PM - MP)/2 with parent
    (PM + MP)/2 = SF (Eq. 11-12).  |NM| <= NUC + PROJ and |CHI| <= SF pointwise."""
    M = oracle_mod.response(A, th, [KI["NUC"], KI["PROJ"], KI["SF"]], P=P, sN=sN, sM=sM, invV=invV)
    return {KI["NM"]: M[0] + M[1], KI["CHI"]: M[2]}


def assert_cross_sections(M_gpu, M_ref, kinds, label="", ref_max=None, parents=None, parent_max=None, signed_misses=None):
    """north_star, literally: relative error <= 1e-3 wherever |oracle| > 1e-6 of the map's own maximum, for every
    kind, the signed ones (NM, CHI) included.

    One clarification only (reading 16 (i)): a signed map that is null by symmetry (max|oracle| <= 1e-9 of
    its parent half-sum NUC + PROJ resp. SF: both sides hold rounding noise, 'its maximum' has no meaning) must stay
    below 1e-6 max(parent) on the GPU.  parents: kind -> parent map at the compared points (None = taken from the rows
    of M_ref).  ref_max / parent_max: maxima taken over a larger map than the points compared (sampled comparisons).

    signed_misses: None = a miss of NM / CHI fails the test like any other.  A list = the fp32-accumulating kernels on
    workloads where DESIGN.md section 7 states that the criterion is NOT guaranteed for the signed kinds: their misses
    are appended as (label, kind, points tested, points failing, worst relative error) and the caller reports them with
    `report_signed_misses` (the test then shows as xfailed, never as passed)."""
    kinds = list(kinds)
    if parents is None:   # derive the parents from the oracle rows themselves when they are there
        parents = {}
        if KI["NUC"] in kinds and KI["PROJ"] in kinds:
            parents[KI["NM"]] = M_ref[kinds.index(KI["NUC"])] + M_ref[kinds.index(KI["PROJ"])]
        if KI["SF"] in kinds:
            parents[KI["CHI"]] = M_ref[kinds.index(KI["SF"])]
    for i, k in enumerate(kinds):
        ref = M_ref[i]
        got = M_gpu[i].astype(np.float64)
        mx = np.abs(ref).max() if ref_max is None else ref_max[i]
        par = parents.get(k)
        if par is not None:
            pmax = np.abs(par).max() if parent_max is None else parent_max[k]
            if np.abs(ref).max() <= NULL_LEVEL * pmax:
                worst = np.abs(got - ref).max()
                assert worst <= XS_FLOOR * pmax, f"{label}: null kind {ni.KINDS[k]}: |gpu| up to {worst:.3e} > 1e-6 x parent max {pmax:.3e}"
                continue
        sel = np.abs(ref) > XS_FLOOR * mx
        if not np.any(sel):
            continue
        rel = np.abs(got[sel] - ref[sel]) / np.abs(ref[sel])
        if rel.max() > XS_RTOL and k in SIGNED and signed_misses is not None:
            signed_misses.append((label, ni.KINDS[k], int(sel.sum()), int((rel > XS_RTOL).sum()), float(rel.max())))
            continue
        assert rel.max() <= XS_RTOL, f"{label}: kind {ni.KINDS[k]}: max rel err {rel.max():.3e} at {sel.sum()} points"


def report_signed_misses(misses):
    """Every other assertion of the test held; the north-star criterion for NM / CHI did not hold everywhere: xfail with
    the measured numbers (DESIGN.md section 7 says where the fp32 kernels cannot guarantee it and why)."""
    if misses:
        pytest.xfail("north_star criterion missed for signed kinds (fp32 accumulation, DESIGN.md section 7): " +
                     "; ".join(f"{lab} {kind}: {bad} of {n} points above 1e-3, worst {w:.2e}" for lab, kind, n, bad, w in misses))


def _oracle_maps(oracle_mod, wl, qy, qz, th, kinds, R=None):
    A, wsum = oracle_mod.amplitudes(wl.pos, wl.N, wl.m, wl.R if R is None else R, qy, qz, offsets=wl.offsets,
                                    centres=wl.centres, return_wsum=True)
    M = oracle_mod.response(A, th, kinds, P=wl.P)
    return A, wsum, M


def _run_full(nms, h, wl, kinds):
    import torch
    nq = wl.grid.n_q
    amp = torch.empty((8, nq), dtype=torch.float32, device="cuda")
    maps = torch.empty((len(kinds), nq), dtype=torch.float32, device="cuda")
    maps2 = torch.empty_like(maps)
    nms.nms_amplitudes(h, wl.grid, amp)
    nms.nms_response(h, kinds, maps)
    nms.nms_compute(h, wl.grid, kinds, maps2)
    nms.nms_synchronize(h)
    assert torch.equal(maps, maps2), "nms_compute and nms_amplitudes+nms_response disagree"
    return amp.cpu().numpy(), maps.cpu().numpy()


# ---------------------------------------------------------------------------------------------------
# C1, C2 at full size, full maps; every kernel variant the grid admits
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["C1", "C2"])
@pytest.mark.parametrize("variant,qt,bases,rec,prec", [(0, 0, 0, 0, 0), (3, 0, 0, 0, 0), (1, 0, 0, 0, 1), (1, 4, 0, 0, 1),
                                                        (1, 8, 0, 0, 1), (1, 0, 0, 0, 2), (1, 4, 0, 0, 0),
                                                        (2, 0, 0, 0, 1), (2, 0, 1, 1, 1), (2, 0, 2, 1, 1), (2, 0, 2, 2, 1),
                                                        (2, 0, 3, 1, 1), (2, 0, 4, 1, 1), (2, 0, 0, 0, 0), (2, 0, 2, 2, 2),
                                                        (2, 16, 0, 0, 1), (2, 16, 0, 0, 0)])
def test_full_config_maps(nms, ctx, oracle_mod, name, variant, qt, bases, rec, prec):
    """variant 0 = automatic (these small problems run the exact fp64 kernel), 3 = exact forced: every kind held to
    the north_star criterion.  1 = the fp32-accumulating direct kernels, 2 = the line-recurrence kernels with `bases`
    exactly evaluated points per 8 by rotations (rec 1) or the three-term recurrence (rec 2) -- qt 16: the 16-point
    kernels large problems get, 2 exact points + three-term (fast) or 1 + rotations (accurate) --, MUFU (prec 1) or
    polynomial (prec 2; prec 0 = automatic, which is 2 here: all 13 kinds are asked for) phasors: amplitudes and every
    kind to the same criterion; a miss of NM / CHI is reported as xfail (C1 and C2 are below the size where the library
    itself would pick an fp32 kernel)."""
    wl = ni.make_config(name)
    kinds = list(ni.ALL_KINDS)
    _upload(nms, ctx, wl)
    nms.nms_set_option(ctx, "variant", variant)
    nms.nms_set_option(ctx, "qt", qt)
    nms.nms_set_option(ctx, "bases", bases)
    nms.nms_set_option(ctx, "recurrence", rec)
    nms.nms_set_option(ctx, "precision", prec)
    A_gpu, M_gpu = _run_full(nms, ctx, wl, kinds)
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    A, wsum, M = _oracle_maps(oracle_mod, wl, qy, qz, th, kinds)
    np.testing.assert_allclose(nms.nms_get_weight_sums(ctx), wsum, rtol=1e-12)
    assert_amplitudes(A_gpu, A, wsum, name)
    misses = [] if variant in (1, 2) else None
    assert_cross_sections(M_gpu, M, kinds, name, signed_misses=misses)
    used = nms.nms_get_info(ctx, "variant_used")
    polar = wl.grid.type == 0
    assert used == {0: 8, 3: 8, 1: 2 if polar else 4, 2: 3 if polar else 5}[variant]
    if variant in (1, 2):
        assert (nms.nms_get_info(ctx, "poly_phasors") != 0) == (prec != 1)
    if variant == 2:
        assert nms.nms_get_info(ctx, "bases") == (bases or (2 if qt == 16 and prec == 1 else 1))
        assert nms.nms_get_info(ctx, "qt") == (qt or 8)
        assert nms.nms_get_info(ctx, "three_term") == (1 if rec == 2 or (rec == 0 and prec == 1) else 0)
    report_signed_misses(misses)


def test_c1_physics_on_gpu(nms, ctx):
    """Uniform M_z sphere (Eq. 60-63): MAG = |F|^2 sin^2 th, SF = |F|^2 sin^2 cos^2, CHI = 0 exactly."""
    wl = ni.make_config("C1")
    _upload(nms, ctx, wl)
    kinds = [KI["NUC"], KI["MAG"], KI["SF"], KI["CHI"]]
    _, M = _run_full(nms, ctx, wl, kinds)
    th = np.tile(wl.grid.u1.astype(np.float64), wl.grid.n0)
    s2, c2 = np.sin(th) ** 2, np.cos(th) ** 2
    big = M[0] > 1e-6 * M[0].max()
    np.testing.assert_allclose(M[1][big], (M[0] * s2)[big], rtol=2e-6, atol=1e-6 * M[0].max() * 1e-6)
    np.testing.assert_allclose(M[2][big], (M[0] * s2 * c2)[big], rtol=2e-5, atol=1e-12 * M[0].max())
    assert np.all(M[3] == 0.0)


# ---------------------------------------------------------------------------------------------------
# reduced C3, C4, C5 (same structure, several tiles and a ragged tail), full maps
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["C3", "C4", "C5"])
@pytest.mark.parametrize("variant,prec", [(0, 0), (1, 1), (2, 1), (1, 2), (2, 0)])
def test_small_config_maps(nms, ctx, oracle_mod, name, variant, prec):
    """Every kernel family on the reduced configs, all 13 kinds at the north_star criterion (variant 0 picks the exact
    kernel at these sizes; a miss of NM / CHI by an fp32 kernel is reported as xfail)."""
    if name == "C3" and variant == 2:
        pytest.skip("C3's |q| is log-spaced: no line recurrence (NMS_E_UNSUPPORTED, see test_error_codes)")
    wl = ni.make_config(name, small=True)
    kinds = list(ni.ALL_KINDS)
    nms.nms_set_option(ctx, "variant", variant)
    nms.nms_set_option(ctx, "precision", prec)
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    rots = wl.rotations if wl.rotations is not None else [wl.R]
    _upload(nms, ctx, wl)
    misses = [] if variant else None
    for R in rots:
        nms.nms_set_rotation(ctx, R)
        A_gpu, M_gpu = _run_full(nms, ctx, wl, kinds)
        A, wsum, M = _oracle_maps(oracle_mod, wl, qy, qz, th, kinds, R=R)
        assert_amplitudes(A_gpu, A, wsum, name)
        assert_cross_sections(M_gpu, M, kinds, name, signed_misses=misses)
        assert (nms.nms_get_info(ctx, "variant_used") == 8) == (variant == 0)
    report_signed_misses(misses)


@pytest.mark.parametrize("gtype", [0, 1])
@pytest.mark.parametrize("n0,qt", [(1, 0), (2, 0), (7, 0), (13, 0), (24, 0), (2, 16), (13, 16), (24, 16), (33, 16)])
def test_recurrence_ragged_lines(nms, ctx, oracle_mod, gtype, n0, qt):
    """Line recurrence on detector lines whose length is not a multiple of the 8 or 16 points a thread owns (and
    shorter than them): the points beyond the edge continue the progression and are never stored.  qt = 16 forces the
    16-point kernels that large problems get (this one is too small to be given them automatically)."""
    rng = np.random.Generator(np.random.Philox(4242))
    W = 3000
    pos = rng.uniform(-40, 40, size=(W, 3)).astype(np.float32)
    N = rng.uniform(0.5, 1.5, size=W).astype(np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    R = ni.rot_z(20.0) @ ni.rot_y(35.0) @ ni.rot_z(10.0)
    if gtype == 0:
        grid = ni.polar_grid(np.linspace(0.02, 1.7, n0) if n0 > 1 else np.array([0.5]), 37)
    else:
        grid = ni.cartesian_grid(np.linspace(-0.9, 1.1, n0) if n0 > 1 else np.array([0.3]), np.linspace(-1.0, 1.0, 37))
    kinds = list(ni.ALL_KINDS)   # a fully incoherent random sample: the signed kinds cross zero all over the detector
    import torch
    nms.nms_set_sample(ctx, _t(pos), _t(N), _t(m), R)
    nms.nms_set_option(ctx, "variant", 2 if n0 > 1 else 1)
    nms.nms_set_option(ctx, "qt", qt)
    amp = torch.empty((8, grid.n_q), dtype=torch.float32, device="cuda")
    maps = torch.empty((len(kinds), grid.n_q), dtype=torch.float32, device="cuda")
    qy, qz, th = oracle_mod.grid_points(grid)
    A, wsum = oracle_mod.amplitudes(pos, N, m, R, qy, qz, return_wsum=True)
    M = oracle_mod.response(A, th, kinds)
    misses = []
    for prec in (1, 0):                                     # fast (three-term, MUFU), then automatic = accurate
        nms.nms_set_option(ctx, "precision", prec)
        nms.nms_amplitudes(ctx, grid, amp)
        nms.nms_response(ctx, kinds, maps)
        nms.nms_synchronize(ctx)
        if n0 > 1:
            assert nms.nms_get_info(ctx, "variant_used") == (3 if gtype == 0 else 5)
            assert nms.nms_get_info(ctx, "qt") == (qt if qt else 8)
        assert (nms.nms_get_info(ctx, "poly_phasors") != 0) == (prec == 0)
        assert_amplitudes(amp.cpu().numpy(), A, wsum, f"ragged n0={n0} precision {prec}")
        assert_cross_sections(maps.cpu().numpy(), M, kinds, f"ragged n0={n0} precision {prec}", signed_misses=misses)
    report_signed_misses(misses)


@pytest.mark.parametrize("gtype", [0, 1])
@pytest.mark.parametrize("n0", [3, 4, 5, 15, 16, 17, 18, 33, 48])
def test_interpolating_kernel_ragged_lines(nms, ctx, oracle_mod, gtype, n0):
    """k_amp_interp (the accurate variant large problems get when the step phase of a line stays below 0.2 cycle):
    every other point of a line is generated, the points in between are sums of their neighbours' h-weighted sets.
    Lines of odd and even length (an even one needs one primary beyond the edge), shorter than, equal to and not a
    multiple of the 16 points a thread covers, polar and Cartesian; amplitudes and all 13 kinds against the oracle.
    A step phase beyond 0.2 cycle is refused when the kernel is required, and falls back when it is not."""
    import torch
    rng = np.random.Generator(np.random.Philox(4243))
    W = 3000
    pos = rng.uniform(-40, 40, size=(W, 3)).astype(np.float32)
    N = rng.uniform(0.5, 1.5, size=W).astype(np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    R = ni.rot_z(20.0) @ ni.rot_y(35.0) @ ni.rot_z(10.0)
    u0 = 0.31 + 0.013 * np.arange(n0)                            # d r_max <= 0.013 * 69.3 = 0.9 rad = 0.14 cycle
    if gtype == 0:
        grid = ni.polar_grid(u0, 37)
    else:
        grid = ni.cartesian_grid(u0 - 0.5, np.linspace(-1.0, 1.0, 37))
    kinds = list(ni.ALL_KINDS)
    nms.nms_set_sample(ctx, _t(pos), _t(N), _t(m), R)
    nms.nms_set_option(ctx, "variant", 2)
    nms.nms_set_option(ctx, "qt", 16)
    nms.nms_set_option(ctx, "precision", 2)
    amp = torch.empty((8, grid.n_q), dtype=torch.float32, device="cuda")
    maps = torch.empty((len(kinds), grid.n_q), dtype=torch.float32, device="cuda")
    qy, qz, th = oracle_mod.grid_points(grid)
    A, wsum = oracle_mod.amplitudes(pos, N, m, R, qy, qz, return_wsum=True)
    M = oracle_mod.response(A, th, kinds)
    misses = []
    for interp in (2, 0, 1):                                     # required, automatic (= used), switched off
        nms.nms_set_option(ctx, "interp", interp)
        amp.fill_(float("nan")); maps.fill_(float("nan"))
        nms.nms_amplitudes(ctx, grid, amp)
        nms.nms_response(ctx, kinds, maps)
        nms.nms_synchronize(ctx)
        assert nms.nms_get_info(ctx, "variant_used") == (3 if gtype == 0 else 5)
        assert nms.nms_get_info(ctx, "interp") == (0 if interp == 1 else 1)
        assert nms.nms_get_info(ctx, "qt") == 16 and nms.nms_get_info(ctx, "poly_phasors") != 0
        assert_amplitudes(amp.cpu().numpy(), A, wsum, f"interp {interp} n0={n0}")
        assert_cross_sections(maps.cpu().numpy(), M, kinds, f"interp {interp} n0={n0}", signed_misses=misses)
    coarse = ni.polar_grid(0.31 + 0.05 * np.arange(n0), 37) if gtype == 0 else \
        ni.cartesian_grid(0.05 * np.arange(n0) - 0.2, np.linspace(-1.0, 1.0, 37))
    nms.nms_set_option(ctx, "interp", 2)
    with pytest.raises(nms.NmsError) as e:
        nms.nms_amplitudes(ctx, coarse, None)
    assert e.value.status == nms.NMS_E_UNSUPPORTED
    nms.nms_set_option(ctx, "interp", 0)
    nms.nms_amplitudes(ctx, coarse, None)
    assert nms.nms_get_info(ctx, "interp") == 0
    report_signed_misses(misses)


# ---------------------------------------------------------------------------------------------------
# C3, C4, C5 at BASELINE.json's full sizes, in the launch configuration bench.py times (automatic
# variant): the full GPU map against the oracle on a seeded subset of detector points; maxima for the
# floors are taken over the GPU's full map
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,n_sample", [("C3", 96), ("C4", 64), ("C5", 64)])
def test_full_size_sampled(nms, ctx, oracle_mod, name, n_sample):
    """All 13 kinds; C4: 6 of its 36 rotations, spread over the scan."""
    import torch
    wl = ni.make_config(name)
    kinds = list(ni.ALL_KINDS)
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    idx = ni.q_subset(wl.grid.n_q, n_sample, 9000 + int(name[1]))
    rots = [wl.rotations[i] for i in (0, 7, 13, 20, 27, 35)] if wl.rotations is not None else [wl.R]
    _upload(nms, ctx, wl)
    nq = wl.grid.n_q
    amp = torch.empty((8, nq), dtype=torch.float32, device="cuda")
    maps = torch.empty((len(kinds), nq), dtype=torch.float32, device="cuda")
    for R in rots:
        nms.nms_set_rotation(ctx, R)
        nms.nms_amplitudes(ctx, wl.grid, amp)
        nms.nms_response(ctx, kinds, maps)
        nms.nms_synchronize(ctx)
        # an fp32-accumulating kernel: direct for C3 (log-spaced |q|), line recurrence for C4 and C5 -- the accurate
        # variant, automatically: the amplitudes are kept for whatever kinds nms_response is asked for
        assert nms.nms_get_info(ctx, "variant_used") == {"C3": 2, "C4": 5, "C5": 3}[name]
        assert nms.nms_get_info(ctx, "poly_phasors") != 0
        A_gpu, M_gpu = amp.cpu().numpy(), maps.cpu().numpy()
        A, wsum = oracle_mod.amplitudes(wl.pos, wl.N, wl.m, R, qy[idx], qz[idx], offsets=wl.offsets,
                                        centres=wl.centres, return_wsum=True)
        M = oracle_mod.response(A, th[idx], kinds, P=wl.P)
        assert_amplitudes(A_gpu[:, idx], A, wsum, name)
        full_max = np.abs(M_gpu.astype(np.float64)).max(axis=1)
        par = parent_maps(oracle_mod, A, th[idx], wl.P)
        # parents' maxima over the full GPU map as well
        pmax = {KI["NM"]: full_max[kinds.index(KI["NUC"])] + full_max[kinds.index(KI["PROJ"])],
                KI["CHI"]: full_max[kinds.index(KI["SF"])]}
        assert_cross_sections(M_gpu[:, idx], M, kinds, name, ref_max=full_max, parents=par, parent_max=pmax)


@pytest.fixture(scope="module")
def c5_full(oracle_mod):
    """The workload C5 and its full-map fp64 reference (exact x-collapse, tests/c5_reference.py); 1-3 minutes of CPU."""
    import c5_reference
    wl = ni.make_config("C5")
    A, wsum, th = c5_reference.full_reference(oracle_mod, wl)
    return wl, A, wsum, th


@pytest.mark.parametrize("precision,interp", [(0, 0), (1, 0), (0, 1)])
def test_c5_full_map_end_to_end(nms, ctx, oracle_mod, c5_full, precision, interp):
    """C5 at full size through the call sequence bench.py times (nms_compute, ring average, c(r), p(r)) against the
    FULL fp64 map of the oracle: all 13 maps at every one of the 262 144 detector points, the amplitudes, the 512-ring
    I(q) (Eq. 30) and c(r), p(r) at 1024 r (Eq. 34-35).
    precision 0: what the library picks itself for C5's 13 kinds -- the accurate variant (polynomial phasors, rotations,
    fp64 sub-accumulation of the nuclear channel; every other point of a line generated, the points in between taken from
    the sums: k_amp_interp), the configuration of the headline bench line: every kind, NM and CHI included, must meet the
    north_star criterion at every point -- and so must the accurate variant that generates all 16 points of a thread
    (interp 1: the interpolating kernel switched off).  precision 1: the fast variant (three-term recurrence, MUFU
    phasors) forced: a miss of NM / CHI is reported as xfail."""
    import torch
    wl, A, wsum, th = c5_full
    kinds = wl.kinds
    M = oracle_mod.response(A, th, kinds, P=wl.P)
    _upload(nms, ctx, wl)
    nms.nms_set_option(ctx, "precision", precision)
    nms.nms_set_option(ctx, "interp", interp)
    nq, nb, nr, nk = wl.grid.n_q, wl.n_bins, len(wl.r), len(kinds)
    f32 = dict(dtype=torch.float32, device="cuda")
    maps, I, qb = torch.empty((nk, nq), **f32), torch.empty((nk, nb), **f32), torch.empty(nb, **f32)
    cnt = torch.empty(nb, dtype=torch.int32, device="cuda")
    c, p = torch.empty((nk, nr), **f32), torch.empty((nk, nr), **f32)
    amp = torch.empty((8, nq), **f32)
    nms.nms_compute(ctx, wl.grid, kinds, maps)
    nms.nms_azimuthal_average(ctx, maps, nk, nb, wl.q_lo, wl.q_hi, I, qb, cnt)
    nms.nms_correlation(ctx, I, qb, cnt, nk, nb, _t(wl.r), c, p)
    nms.nms_amplitudes(ctx, wl.grid, amp)
    nms.nms_synchronize(ctx)
    assert nms.nms_get_info(ctx, "variant_used") == 3
    assert (nms.nms_get_info(ctx, "poly_phasors") != 0) == (precision == 0)
    assert nms.nms_get_info(ctx, "interp") == (1 if precision == 0 and interp == 0 else 0)
    np.testing.assert_allclose(nms.nms_get_weight_sums(ctx), wsum, rtol=1e-12)
    assert_amplitudes(amp.cpu().numpy(), A, wsum, "C5 full map")
    misses = [] if precision == 1 else None
    assert_cross_sections(maps.cpu().numpy(), M, kinds, "C5 full map", signed_misses=misses)
    # 1-D outputs.  north_star states a criterion for the 2-D cross sections only; what it implies for a ring mean and
    # for its Fourier-Bessel transform follows by the triangle inequality: maps within 1e-3
    # relative above 1e-6 of their maximum give |dI(q_i)| <= 1e-3 (mean_j |f(q_i, th_j)| + 1e-6 max|f|), and
    # |dc(r)| <= (1 / 2 pi^2) sum_i wq_i q_i^2 |j0(q_i r)| tol_I(q_i), |dp| = r^2 |dc|.  (A relative criterion on I, c, p
    # themselves is meaningless where they vanish: the ring mean of the chiral map is zero by symmetry, L183, and
    # c(r) of every kind oscillates about zero at large r.)  Valid for all kinds, signed ones included.
    n0, n1 = wl.grid.n0, wl.grid.n1
    I_ref = oracle_mod.azimuthal_polar(M, n0, n1)
    assert np.array_equal(cnt.cpu().numpy(), np.full(nb, n1, dtype=np.int32))
    tol_I = 1e-3 * (np.abs(M).reshape(nk, n0, n1).mean(axis=2) + 1e-6 * np.abs(M).max(axis=1)[:, None])
    dI = np.abs(I.cpu().numpy().astype(np.float64) - I_ref)
    assert np.all(dI <= tol_I), f"C5 I(q): worst |dI| / tol = {(dI / tol_I).max():.3f}"
    q = wl.grid.u0.astype(np.float64)
    r = wl.r.astype(np.float64)
    wq = np.empty(n0)
    wq[0], wq[-1] = 0.5 * (q[1] - q[0]), 0.5 * (q[-1] - q[-2])
    wq[1:-1] = 0.5 * (q[2:] - q[:-2])
    x = q[None, :] * r[:, None]
    j0 = np.where(np.abs(x) < 1e-4, 1.0 - x * x / 6.0, np.sin(x) / np.where(x == 0.0, 1.0, x))
    tol_c = (tol_I * (wq * q * q)[None, :]) @ np.abs(j0).T / (2.0 * np.pi ** 2)          # [nk, nr]
    c_ref, p_ref = oracle_mod.correlation(I_ref, q, wl.r)
    dc = np.abs(c.cpu().numpy().astype(np.float64) - c_ref)
    dp = np.abs(p.cpu().numpy().astype(np.float64) - p_ref)
    assert np.all(dc <= tol_c + 1e-7 * np.abs(c_ref)), f"C5 c(r): worst |dc| / tol = {(dc / tol_c).max():.3f}"
    assert np.all(dp <= tol_c * r[None, :] ** 2 + 1e-7 * np.abs(p_ref)), "C5 p(r)"
    # for the record: how close the 1-D outputs actually are, relative to their own maxima
    print("C5 1-D outputs: max |dI| / max|I| per kind", (dI.max(axis=1) / np.abs(I_ref).max(axis=1)).max(),
          "max |dc| / max|c|", (dc.max(axis=1) / np.abs(c_ref).max(axis=1)).max(),
          "worst |dI| / tol", (dI / tol_I).max(), "worst |dc| / tol", (dc / tol_c).max())
    report_signed_misses(misses)


@pytest.mark.parametrize("chunks", [0, 7])
def test_c3_full_size_split_sampled(nms, ctx, oracle_mod, chunks):
    """Full C3 (K = 1000 objects of 4224 cells) through nms_form_factor_split, the call bench.py times: total AND form
    (Eq. 49-50) of the config's four kinds against oracle.form_factor_split on a seeded subset of detector
    points; automatic chunking (object-boundary table) and a forced 7-chunk split."""
    import torch
    wl = ni.make_config("C3")
    kinds = wl.kinds
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    idx = ni.q_subset(wl.grid.n_q, 64, 9003)
    tot_ref, form_ref = oracle_mod.form_factor_split(wl.pos, wl.N, wl.m, wl.offsets, kinds, qy[idx], qz[idx], th[idx], R=wl.R,
                                                     centres=wl.centres, P=wl.P)
    _upload(nms, ctx, wl)
    nms.nms_set_option(ctx, "chunks", chunks)
    tot = torch.empty((len(kinds), wl.grid.n_q), dtype=torch.float32, device="cuda")
    form = torch.empty_like(tot)
    nms.nms_form_factor_split(ctx, wl.grid, kinds, tot, form)
    nms.nms_synchronize(ctx)
    assert nms.nms_get_info(ctx, "variant_used") == 2            # the fp32 direct kernel, per-particle instantiation
    if chunks:
        assert nms.nms_get_info(ctx, "n_chunks") == chunks
    t, f = tot.cpu().numpy(), form.cpu().numpy()
    assert_cross_sections(t[:, idx], tot_ref, kinds, "C3 split total", ref_max=np.abs(t.astype(np.float64)).max(axis=1))
    assert_cross_sections(f[:, idx], form_ref, kinds, "C3 split form", ref_max=np.abs(f.astype(np.float64)).max(axis=1))
    # the ordinary path gives the same total
    maps = torch.empty_like(tot)
    nms.nms_compute(ctx, wl.grid, kinds, maps)
    nms.nms_synchronize(ctx)
    assert_cross_sections(maps.cpu().numpy()[:, idx], tot_ref, kinds, "C3 ordinary total",
                          ref_max=np.abs(t.astype(np.float64)).max(axis=1))


def test_form_factor_split_small(nms, ctx, oracle_mod):
    """Eq. 49-50: total = B(sum A_p), form = sum B(A_p); with and without separate object centres."""
    import torch
    for sep in (False, True):
        wl = ni.config_c3(K=7, n_q=21, n_theta=40, separate_centres=sep)
        kinds = list(ni.ALL_KINDS)
        _upload(nms, ctx, wl)
        qy, qz, th = oracle_mod.grid_points(wl.grid)
        tot_ref, form_ref = oracle_mod.form_factor_split(wl.pos, wl.N, wl.m, wl.offsets, kinds, qy, qz, th, R=wl.R,
                                                         centres=wl.centres, P=wl.P)
        misses = []
        for variant, prec in ((0, 0), (1, 1), (1, 2)):   # exact kernel (automatic at this size), fp32 direct kernel, MUFU / polynomial
            nms.nms_set_option(ctx, "variant", variant)
            nms.nms_set_option(ctx, "precision", prec)
            for chunks in (0, 1, 3):
                nms.nms_set_option(ctx, "chunks", chunks)
                tot = torch.empty((len(kinds), wl.grid.n_q), dtype=torch.float32, device="cuda")
                form = torch.empty_like(tot)
                nms.nms_form_factor_split(ctx, wl.grid, kinds, tot, form)
                nms.nms_synchronize(ctx)
                assert nms.nms_get_info(ctx, "variant_used") == (2 if variant else 8)
                sm = misses if variant else None
                assert_cross_sections(tot.cpu().numpy(), tot_ref, kinds, f"split total v{variant}", signed_misses=sm)
                assert_cross_sections(form.cpu().numpy(), form_ref, kinds, f"split form v{variant}", signed_misses=sm)
            nms.nms_set_option(ctx, "chunks", 0)
            # the ordinary path gives the same total
            maps = torch.empty_like(tot)
            nms.nms_compute(ctx, wl.grid, kinds, maps)
            nms.nms_synchronize(ctx)
            assert_cross_sections(maps.cpu().numpy(), tot_ref, kinds, "ordinary total", signed_misses=sm)
        nms.nms_set_option(ctx, "variant", 0)
        nms.nms_set_option(ctx, "precision", 0)
    report_signed_misses(misses)


@pytest.mark.parametrize("gtype,n1", [(0, 40), (0, 128), (1, 37)])
def test_form_factor_split_line_recurrence(nms, ctx, oracle_mod, gtype, n1):
    """The per-particle instantiation of the line-recurrence kernels (equally spaced |q| or q_z): total and form of the
    positive kinds; n1 = 128 also runs the block-uniform instantiation of the polar three-term kernel in nms_compute."""
    import torch
    wl = ni.config_c3(K=5, n_q=24, n_theta=n1)
    grid = ni.polar_grid(np.linspace(0.02, 1.9, 24), n1) if gtype == 0 else \
        ni.cartesian_grid(np.linspace(-1.6, 1.7, 24), np.linspace(-1.5, 1.5, n1))
    kinds = [KI[k] for k in ("NUC", "MAG", "UNPOL", "PROJ", "SF")]
    _upload(nms, ctx, wl)
    qy, qz, th = oracle_mod.grid_points(grid)
    tot_ref, form_ref = oracle_mod.form_factor_split(wl.pos, wl.N, wl.m, wl.offsets, kinds, qy, qz, th, R=wl.R,
                                                     centres=wl.centres, P=wl.P)
    tot = torch.empty((len(kinds), grid.n_q), dtype=torch.float32, device="cuda")
    form = torch.empty_like(tot)
    maps = torch.empty_like(tot)
    for rec, prec in ((0, 0), (1, 0), (0, 2)):
        nms.nms_set_option(ctx, "variant", 2)
        nms.nms_set_option(ctx, "recurrence", rec)
        nms.nms_set_option(ctx, "precision", prec)
        nms.nms_form_factor_split(ctx, grid, kinds, tot, form)
        nms.nms_synchronize(ctx)
        assert nms.nms_get_info(ctx, "variant_used") == (3 if gtype == 0 else 5)
        assert_cross_sections(tot.cpu().numpy(), tot_ref, kinds, f"split recurrence total {rec} {prec}")
        assert_cross_sections(form.cpu().numpy(), form_ref, kinds, f"split recurrence form {rec} {prec}")
        nms.nms_compute(ctx, grid, kinds, maps)
        nms.nms_synchronize(ctx)
        assert_cross_sections(maps.cpu().numpy(), tot_ref, kinds, f"recurrence ordinary total {rec} {prec}")


def test_form_factor_split_uneven_objects(nms, ctx, oracle_mod):
    """Objects of very different sizes (1 cell .. > 1 tile), one of them empty."""
    import torch
    rng = np.random.Generator(np.random.Philox(77))
    sizes = [1, 0, 1500, 7, 1024, 2049, 33]
    W = sum(sizes)
    offsets = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    pos = rng.uniform(-30, 30, size=(W, 3)).astype(np.float32)
    N = rng.uniform(0.5, 1.5, size=W).astype(np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    cen = rng.uniform(-100, 100, size=(len(sizes), 3)).astype(np.float32)
    R = ni.rotation_alpha_beta(20.0, 50.0)
    grid = ni.polar_grid(0.02 * 1.3 ** np.arange(13), 24)
    kinds = list(ni.ALL_KINDS)
    nms.nms_set_sample(ctx, _t(pos), _t(N), _t(m), R)
    nms.nms_set_particles(ctx, offsets, _t(cen))
    qy, qz, th = oracle_mod.grid_points(grid)
    tot_ref, form_ref = oracle_mod.form_factor_split(pos, N, m, offsets, kinds, qy, qz, th, R=R, centres=cen)
    tot = torch.empty((len(kinds), grid.n_q), dtype=torch.float32, device="cuda")
    form = torch.empty_like(tot)
    misses = []
    for variant in (0, 1):                                   # exact kernel, then the fp32 per-particle kernel
        nms.nms_set_option(ctx, "variant", variant)
        nms.nms_form_factor_split(ctx, grid, kinds, tot, form)
        nms.nms_synchronize(ctx)
        assert nms.nms_get_info(ctx, "variant_used") == (2 if variant else 8)
        sm = misses if variant else None
        assert_cross_sections(tot.cpu().numpy(), tot_ref, kinds, "uneven total", signed_misses=sm)
        assert_cross_sections(form.cpu().numpy(), form_ref, kinds, "uneven form", signed_misses=sm)
    report_signed_misses(misses)


# ---------------------------------------------------------------------------------------------------
# azimuthal average and correlation: pass-isolated (oracle pass on the GPU's own maps) and end to end
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["C1", "C2"])
def test_azimuthal_and_correlation(nms, ctx, oracle_mod, name):
    import torch
    wl = ni.make_config(name)
    kinds = wl.kinds
    _upload(nms, ctx, wl)
    nq = wl.grid.n_q
    maps = torch.empty((len(kinds), nq), dtype=torch.float32, device="cuda")
    nms.nms_compute(ctx, wl.grid, kinds, maps)
    nb = wl.n_bins
    I = torch.empty((len(kinds), nb), dtype=torch.float32, device="cuda")
    qb = torch.empty(nb, dtype=torch.float32, device="cuda")
    cnt = torch.empty(nb, dtype=torch.int32, device="cuda")
    nms.nms_azimuthal_average(ctx, maps, len(kinds), nb, wl.q_lo, wl.q_hi, I, qb, cnt)
    nms.nms_synchronize(ctx)
    maps_h, I_h, qb_h, cnt_h = maps.cpu().numpy(), I.cpu().numpy(), qb.cpu().numpy(), cnt.cpu().numpy()
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    if wl.grid.type == 0:
        I_iso = oracle_mod.azimuthal_polar(maps_h, wl.grid.n0, wl.grid.n1)
        cnt_ref = np.full(nb, wl.grid.n1, dtype=np.int32)
        q_ref = wl.grid.u0.astype(np.float64)
    else:
        I_iso, cnt_ref = oracle_mod.azimuthal_hist(maps_h, qy, qz, nb, wl.q_lo, wl.q_hi)
        q_ref = oracle_mod.hist_bin_centres(nb, wl.q_lo, wl.q_hi)
    assert np.array_equal(cnt_h, cnt_ref)                       # integer work: bit exact
    np.testing.assert_allclose(qb_h, q_ref, rtol=1e-6)
    scale = np.abs(I_iso).max(axis=1, keepdims=True)
    assert np.all(np.abs(I_h - I_iso) <= 2e-7 * scale + 1e-6 * np.abs(I_iso))   # pass-isolated: fp32 output rounding only
    # end to end against the oracle's own maps
    A, wsum, M = _oracle_maps(oracle_mod, wl, qy, qz, th, kinds)
    I_ref = oracle_mod.azimuthal_polar(M, wl.grid.n0, wl.grid.n1) if wl.grid.type == 0 else oracle_mod.azimuthal_hist(M, qy, qz, nb, wl.q_lo, wl.q_hi)[0]
    assert_cross_sections(I_h, I_ref, kinds, name + " I(q)")
    # correlation function
    r = wl.r if wl.r is not None else np.linspace(0.0, 25.0, 64).astype(np.float32)
    r_d = _t(r)
    c = torch.empty((len(kinds), len(r)), dtype=torch.float32, device="cuda")
    p = torch.empty_like(c)
    nms.nms_correlation(ctx, I, qb, cnt, len(kinds), nb, r_d, c, p)
    nms.nms_synchronize(ctx)
    c_iso, p_iso = oracle_mod.correlation(I_h, qb_h, r, count=cnt_h)
    for got, want in ((c.cpu().numpy(), c_iso), (p.cpu().numpy(), p_iso)):
        sc = np.abs(want).max(axis=1, keepdims=True)
        assert np.all(np.abs(got - want) <= 3e-7 * sc + 1e-6 * np.abs(want))
    c_ref, p_ref = oracle_mod.correlation(I_ref, q_ref, r, count=cnt_ref)
    assert_cross_sections(c.cpu().numpy(), c_ref, kinds, name + " c(r)")
    assert_cross_sections(p.cpu().numpy(), p_ref, kinds, name + " p(r)")


@pytest.mark.parametrize("name,small,k_max", [("C1", False, 6), ("C5", True, 8), ("C3", True, 0), ("C5", True, 63)])
def test_modal_decomposition(nms, ctx, oracle_mod, name, small, k_max):
    """f-2, Eq. 31-33: pass-isolated (oracle applied to the GPU's own maps: fp32 output rounding only) and end to
    end against the oracle's maps; the chiral map's sine harmonics are the reason the paper has this pass (L183)."""
    import torch
    wl = ni.make_config(name, small=small)
    kinds = list(ni.ALL_KINDS)
    _upload(nms, ctx, wl)
    n0, n1, nk, nm = wl.grid.n0, wl.grid.n1, k_max + 1, len(kinds)
    maps = torch.empty((nm, wl.grid.n_q), dtype=torch.float32, device="cuda")
    nms.nms_compute(ctx, wl.grid, kinds, maps)
    Is = torch.empty((nm, nk, n0), dtype=torch.float32, device="cuda")
    Ic = torch.empty_like(Is)
    a = torch.empty((nm, 2, nk), dtype=torch.float32, device="cuda")
    A = torch.empty_like(a)
    nms.nms_modal_decomposition(ctx, maps, nm, k_max, Is, Ic, a, A)
    nms.nms_synchronize(ctx)
    maps_h = maps.cpu().numpy()
    rIs, rIc, ras, rac, rAs, rAc = oracle_mod.modal(maps_h, n0, n1, wl.grid.u1, k_max)
    scale = np.abs(maps_h).max(axis=1)[:, None, None]              # |I_k| <= 2 max|f|
    for got, want in ((Is.cpu().numpy(), rIs), (Ic.cpu().numpy(), rIc)):
        assert np.all(np.abs(got - want) <= 1e-6 * np.abs(want) + 1e-9 * scale)
    ascale = np.maximum(np.abs(ras), np.abs(rac)).max(axis=1)[:, None]
    a_h, A_h = a.cpu().numpy(), A.cpu().numpy()
    assert np.all(np.abs(a_h[:, 0] - ras) <= 1e-6 * np.abs(ras) + 1e-9 * ascale)
    assert np.all(np.abs(a_h[:, 1] - rac) <= 1e-6 * np.abs(rac) + 1e-9 * ascale)
    assert np.all(np.abs(A_h[:, 0] - rAs) <= 2e-7) and np.all(np.abs(A_h[:, 1] - rAc) <= 2e-7)   # |A| <= 1
    # end to end: harmonics of the oracle's own maps; an absolute criterion on the scale of the map
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    _, _, M = _oracle_maps(oracle_mod, wl, qy, qz, th, kinds)
    eIs, eIc, eas, eac, eAs, eAc = oracle_mod.modal(M, n0, n1, wl.grid.u1, k_max)
    ring_scale = np.abs(M).reshape(nm, n0, n1).max(axis=2)[:, None, :]   # per ring: |I_k(q_i)| <= 2 max_j |f(q_i, .)|
    fp32 = nms.nms_get_info(ctx, "variant_used") != 8
    # a harmonic is a mean over the ring with weights of modulus <= 2: maps that are pointwise within the north-star
    # 1e-3 (MUFU kernels; the exact kernel leaves only the fp32 rounding of the stored maps) give harmonics within
    # 2 tol max_j |f(q_i, theta_j)|
    tol = 1e-3 if fp32 else 2e-7
    assert np.all(np.abs(Ic.cpu().numpy() - eIc) <= 2 * tol * ring_scale)
    assert np.all(np.abs(Is.cpu().numpy() - eIs) <= 2 * tol * ring_scale)
    np.testing.assert_allclose(A_h[:, 1, 0], eAc[:, 0], rtol=1e-3, atol=1e-6)


def test_modal_decomposition_errors(nms, ctx):
    import torch
    wl = ni.make_config("C2")                                      # Cartesian detector: no rings
    _upload(nms, ctx, wl)
    maps = torch.empty((1, wl.grid.n_q), dtype=torch.float32, device="cuda")
    out = torch.empty((1, 2, 3), dtype=torch.float32, device="cuda")
    with pytest.raises(nms.NmsError) as e:
        nms.nms_modal_decomposition(ctx, maps, 1, 2, None, None, out, None)
    assert e.value.status == nms.NMS_E_STATE                       # no grid yet
    nms.nms_compute(ctx, wl.grid, [0], maps)
    with pytest.raises(nms.NmsError) as e:
        nms.nms_modal_decomposition(ctx, maps, 1, 2, None, None, out, None)
    assert e.value.status == nms.NMS_E_UNSUPPORTED
    wl = ni.make_config("C1")
    _upload(nms, ctx, wl)
    maps = torch.empty((1, wl.grid.n_q), dtype=torch.float32, device="cuda")
    nms.nms_compute(ctx, wl.grid, [0], maps)
    for bad in (-1, 64):
        with pytest.raises(nms.NmsError) as e:
            nms.nms_modal_decomposition(ctx, maps, 1, bad, None, None, out, None)
        assert e.value.status == nms.NMS_E_ARG
    with pytest.raises(nms.NmsError) as e:
        nms.nms_modal_decomposition(ctx, maps, 1, 2, None, None, None, None)
    assert e.value.status == nms.NMS_E_ARG


@pytest.mark.parametrize("variant", [0, 1, 2])
def test_correlation_2d(nms, ctx, oracle_mod, variant):
    """f-1, Eq. 36: C(rho, alpha) of the GPU's own maps (pass-isolated) against the oracle; the criterion is the
    north-star amplitude criterion of the underlying Fourier sum, |dC| <= 1e-5 sum_p |w_p| with w_p = f q wq dtheta.
    The chiral-type odd map gives a purely imaginary C, the even ones a real C (checked on the oracle side)."""
    import torch
    wl = ni.make_config("C5", small=True)
    kinds = [KI["UNPOL"], KI["SF"], KI["CHI"]]
    _upload(nms, ctx, wl)
    n0, n1 = wl.grid.n0, wl.grid.n1
    maps = torch.empty((len(kinds), wl.grid.n_q), dtype=torch.float32, device="cuda")
    nms.nms_compute(ctx, wl.grid, kinds, maps)
    rgrid = ni.polar_grid(np.linspace(0.0, 30.0, 21 if variant != 2 else 24), 36)
    re = torch.empty(rgrid.n_q, dtype=torch.float32, device="cuda")
    im = torch.empty_like(re)
    maps_h = maps.cpu().numpy()
    q64 = wl.grid.u0.astype(np.float64)
    wq = np.empty(n0)
    wq[0], wq[-1] = 0.5 * (q64[1] - q64[0]), 0.5 * (q64[-1] - q64[-2])
    wq[1:-1] = 0.5 * (q64[2:] - q64[:-2])
    nms.nms_set_option(ctx, "variant", variant)
    for i in range(len(kinds)):
        nms.nms_correlation_2d(ctx, maps[i], rgrid, re, im)
        nms.nms_synchronize(ctx)
        if variant == 0:
            assert nms.nms_get_info(ctx, "corr2d_variant") == 8        # small problem: exact kernel
        if variant == 2:
            assert nms.nms_get_info(ctx, "corr2d_variant") == 3        # rho is an arithmetic progression: recurrence
        rre, rim = oracle_mod.correlation_2d(maps_h[i], wl.grid.u0, wl.grid.u1, rgrid.u0, rgrid.u1)
        sw = float((np.abs(maps_h[i].astype(np.float64)).reshape(n0, n1) * (q64 * wq)[:, None]).sum() * 2 * np.pi / n1)
        tol = (1e-5 if variant else 2e-7) * sw
        assert np.abs(re.cpu().numpy().reshape(rgrid.n0, rgrid.n1) - rre).max() <= tol, ni.KINDS[kinds[i]]
        assert np.abs(im.cpu().numpy().reshape(rgrid.n0, rgrid.n1) - rim).max() <= tol, ni.KINDS[kinds[i]]
    nms.nms_set_option(ctx, "variant", 0)
    # the detector grid, the sample and the stored amplitudes of the context are untouched
    maps2 = torch.empty_like(maps)
    nms.nms_compute(ctx, wl.grid, kinds, maps2)
    nms.nms_synchronize(ctx)
    assert torch.equal(maps, maps2)
    I = torch.empty((len(kinds), n0), dtype=torch.float32, device="cuda")
    nms.nms_azimuthal_average(ctx, maps, len(kinds), n0, 0.0, 0.0, I)
    nms.nms_synchronize(ctx)
    np.testing.assert_allclose(I.cpu().numpy(), oracle_mod.azimuthal_polar(maps_h, n0, n1), rtol=2e-6, atol=1e-6 * np.abs(maps_h).max())


def test_correlation_2d_errors(nms, ctx):
    import torch
    wl = ni.make_config("C2")
    _upload(nms, ctx, wl)
    maps = torch.empty((1, wl.grid.n_q), dtype=torch.float32, device="cuda")
    out = torch.empty(8, dtype=torch.float32, device="cuda")
    rgrid = ni.polar_grid(np.linspace(0.0, 1.0, 2), 4)
    with pytest.raises(nms.NmsError) as e:
        nms.nms_correlation_2d(ctx, maps[0], rgrid, out, None)
    assert e.value.status == nms.NMS_E_STATE
    nms.nms_compute(ctx, wl.grid, [0], maps)
    with pytest.raises(nms.NmsError) as e:
        nms.nms_correlation_2d(ctx, maps[0], rgrid, out, None)
    assert e.value.status == nms.NMS_E_UNSUPPORTED                  # Cartesian detector
    wl = ni.make_config("C1")
    _upload(nms, ctx, wl)
    maps = torch.empty((1, wl.grid.n_q), dtype=torch.float32, device="cuda")
    nms.nms_compute(ctx, wl.grid, [0], maps)
    with pytest.raises(nms.NmsError) as e:
        nms.nms_correlation_2d(ctx, maps[0], ni.cartesian_grid(np.zeros(2), np.zeros(2)), out, None)
    assert e.value.status == nms.NMS_E_ARG
    with pytest.raises(nms.NmsError) as e:
        nms.nms_correlation_2d(ctx, maps[0], rgrid, None, None)
    assert e.value.status == nms.NMS_E_ARG


@pytest.mark.parametrize("which", ["nuclear_only", "magnetic_only"])
@pytest.mark.parametrize("variant", [1, 2, 3])
def test_activation_switches(nms, ctx, oracle_mod, which, variant):
    """L242: a sample without moments (m NULL: the one-channel kernel instantiation) or without nuclear weights
    (N NULL); the absent amplitudes must be exactly zero."""
    import torch
    wl = ni.make_config("C5", small=True)
    N, m = (wl.N, None) if which == "nuclear_only" else (None, wl.m)
    kinds = [KI["NUC"], KI["MAG"], KI["UNPOL"], KI["SF"]]
    nms.nms_set_sample(ctx, _t(wl.pos), _t(N), _t(m), wl.R)
    nms.nms_set_option(ctx, "variant", variant)
    if which == "nuclear_only" and variant == 2:
        nms.nms_set_option(ctx, "qt", 16)                          # the 16-points-per-thread one-channel recurrence
    amp = torch.empty((8, wl.grid.n_q), dtype=torch.float32, device="cuda")
    maps = torch.empty((len(kinds), wl.grid.n_q), dtype=torch.float32, device="cuda")
    nms.nms_amplitudes(ctx, wl.grid, amp)
    nms.nms_response(ctx, kinds, maps)
    nms.nms_synchronize(ctx)
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    A, wsum = oracle_mod.amplitudes(wl.pos, N, m, wl.R, qy, qz, return_wsum=True)
    M = oracle_mod.response(A, th, kinds, P=wl.P)
    assert_amplitudes(amp.cpu().numpy(), A, wsum, which)
    if which == "nuclear_only" and variant == 2:
        assert nms.nms_get_info(ctx, "qt") == 16
    got = maps.cpu().numpy()
    live = [0, 2] if which == "nuclear_only" else [1, 2, 3]
    assert_cross_sections(got[live], M[live], [kinds[i] for i in live], which)
    dead = [i for i in range(len(kinds)) if i not in live]
    assert np.all(got[dead] == 0.0)


@pytest.mark.parametrize("name,small", [("C2", False), ("C5", True)])
def test_cross_spectra(nms, ctx, oracle_mod, name, small):
    """f-4, Eq. 51-52: G_ab = invV sM^2 M~_a M~_b^* from the stored amplitudes, with scales; each component within
    1e-3 relative above 1e-6 of the largest |G| (the north-star cross-section criterion), exact kernel and MUFU kernel."""
    import torch
    wl = ni.make_config(name, small=small)
    _upload(nms, ctx, wl)
    sM, invV = 2.5, 1e-3
    nms.nms_set_scales(ctx, 1.0, sM, invV)
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    A = oracle_mod.amplitudes(wl.pos, wl.N, wl.m, wl.R, qy, qz)
    rGR, rGI = oracle_mod.cross_spectra(A, sM=sM, invV=invV)
    gmax = np.abs(rGR).max()
    GR = torch.empty((9, wl.grid.n_q), dtype=torch.float32, device="cuda")
    GI = torch.empty_like(GR)
    with pytest.raises(nms.NmsError) as e:
        nms.nms_cross_spectra(ctx, GR, GI)
    assert e.value.status == nms.NMS_E_STATE                       # no amplitudes yet
    worst = []
    for variant in (0, 1):
        nms.nms_set_option(ctx, "variant", variant)
        nms.nms_amplitudes(ctx, wl.grid, None)
        nms.nms_cross_spectra(ctx, GR, GI)
        nms.nms_synchronize(ctx)
        floor = 1e-6 * gmax                                        # of the largest |G|: the off-diagonal components are signed
        for got, ref in ((GR.cpu().numpy(), rGR), (GI.cpu().numpy(), rGI)):
            sel = np.abs(ref) > floor
            rel = np.abs(got[sel] - ref[sel]) / np.abs(ref[sel])
            if variant == 0 or rel.max() <= 1e-3:
                assert rel.max() <= 1e-3
            else:
                worst.append(f"{name} fp32 kernel: {(rel > 1e-3).sum()} of {sel.sum()} components above 1e-3, worst {rel.max():.2e}")
    with pytest.raises(nms.NmsError) as e:
        nms.nms_cross_spectra(ctx, None, None)
    assert e.value.status == nms.NMS_E_ARG
    if worst:
        pytest.xfail("; ".join(worst))


def test_bench_line_sharded_step_matches_unsharded(nms):
    """bench.py --shard lines on one GPU: the two rank shares of the reduced C5 detector are run one after the
    other (a stand-in process group whose all-gather returns the shares computed so far), and the assembled maps,
    I(q) and c(r), p(r) must equal the unsharded step bit for bit (same kernels, same per-point arithmetic)."""
    import sys, os, torch
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    wl = ni.make_config("C5", small=True)
    ref = bench.Runner(nms, wl, 0)
    nms.nms_set_option(ref.h, "variant", 1)
    ref.step_device()
    nms.nms_synchronize(ref.h)
    world = 2

    class StandIn:                      # all_gather over shares that were computed sequentially on this one GPU
        def __init__(self):
            self.store = {}
            self.rank = 0
        def all_gather(self, parts, pad):
            self.store[self.rank] = pad.clone()
            for r in range(world):
                parts[r].copy_(self.store.get(r, torch.zeros_like(pad)))

    dist = StandIn()
    maps = torch.empty_like(ref.maps)
    c_last = p_last = None
    for rank in (0, 1):
        dist.rank = rank
        part, i0, i1 = bench.shard_workload(wl, world, rank)
        run = bench.Runner(nms, part, 0, shard=(wl, world, rank, dist))
        nms.nms_set_option(run.h, "variant", 1)
        run.step_device()
        nms.nms_synchronize(run.h)
        maps[:, i0 * wl.grid.n1:i1 * wl.grid.n1] = run.maps
        assert torch.equal(run.I, ref.I[:, i0:i1])
        c_last, p_last = run.c.clone(), run.p.clone()
        run.close()
    assert torch.equal(maps, ref.maps)
    assert torch.equal(c_last, ref.c) and torch.equal(p_last, ref.p)     # the last rank saw every ring
    ref.close()


def test_histogram_on_polar_grid_and_empty_bins(nms, ctx, oracle_mod):
    import torch
    wl = ni.make_config("C1")
    _upload(nms, ctx, wl)
    kinds = [KI["NUC"], KI["NM"]]
    maps = torch.empty((2, wl.grid.n_q), dtype=torch.float32, device="cuda")
    nms.nms_compute(ctx, wl.grid, kinds, maps)
    nb = 200                                                       # finer than the 64 rings: many empty bins
    I = torch.empty((2, nb), dtype=torch.float32, device="cuda")
    cnt = torch.empty(nb, dtype=torch.int32, device="cuda")
    nms.nms_azimuthal_average(ctx, maps, 2, nb, 0.5, 2.0, I, None, cnt)
    nms.nms_synchronize(ctx)
    qy, qz, _ = oracle_mod.grid_points(wl.grid)
    I_ref, cnt_ref = oracle_mod.azimuthal_hist(maps.cpu().numpy(), qy, qz, nb, 0.5, 2.0)
    assert np.array_equal(cnt.cpu().numpy(), cnt_ref)
    assert (cnt_ref == 0).sum() > 50
    np.testing.assert_allclose(I.cpu().numpy(), I_ref, rtol=2e-6, atol=0)


# ---------------------------------------------------------------------------------------------------
# edge cases
# ---------------------------------------------------------------------------------------------------
def test_list_grid_with_q_zero_gives_weight_sums(nms, ctx):
    """F(0) = sum w (north_star) through the GPU path; theta(0,0) = 0 (reading 5)."""
    import torch
    rng = np.random.Generator(np.random.Philox(5))
    W = 3001
    pos = rng.normal(scale=20, size=(W, 3)).astype(np.float32)
    N = rng.normal(size=W).astype(np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    R = ni.rotation_alpha_beta(10.0, 20.0)
    nms.nms_set_sample(ctx, _t(pos), _t(N), _t(m), R)
    grid = ni.list_grid(np.zeros(3), np.zeros(3))
    amp = torch.empty((8, 3), dtype=torch.float32, device="cuda")
    nms.nms_amplitudes(ctx, grid, amp)
    nms.nms_synchronize(ctx)
    a = amp.cpu().numpy().astype(np.float64)
    ms = R @ m.astype(np.float64).sum(axis=0)
    want = np.array([N.astype(np.float64).sum(), 0, ms[0], 0, ms[1], 0, ms[2], 0])
    wsum = nms.nms_get_weight_sums(ctx)
    for j in range(3):
        assert np.all(np.abs(a[:, j] - want) <= 1e-6 * np.repeat(wsum, 2) + 1e-30)


@pytest.mark.parametrize("W", [1, 2, 7, 8, 9, 1023, 1024, 1025, 2055])
def test_ragged_cell_counts(nms, ctx, oracle_mod, W):
    import torch
    rng = np.random.Generator(np.random.Philox(100 + W))
    pos = rng.uniform(-15, 15, size=(W, 3)).astype(np.float32)
    N = rng.uniform(-1, 1, size=W).astype(np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    nms.nms_set_sample(ctx, _t(pos), _t(N), _t(m), None)
    grid = ni.polar_grid(np.linspace(0.05, 2.0, 19), 37)              # 19 rings: ragged against QT = 4, 8
    qy, qz, th = oracle_mod.grid_points(grid)
    A, wsum = oracle_mod.amplitudes(pos, N, m, None, qy, qz, return_wsum=True)
    amp = torch.empty((8, grid.n_q), dtype=torch.float32, device="cuda")
    # partial tiles of 1 ... 9 cells and tails behind full tiles through the bulk-copy / mbarrier kernels: direct with
    # 4 and 8 points per thread, MUFU and polynomial phasors, the line recurrence, and the exact kernel
    for variant, qt, prec, used in ((1, 4, 1, 2), (1, 8, 1, 2), (1, 8, 2, 2), (2, 0, 1, 3), (2, 0, 0, 3), (0, 0, 0, 8)):
        nms.nms_set_option(ctx, "variant", variant)
        nms.nms_set_option(ctx, "qt", qt)
        nms.nms_set_option(ctx, "precision", prec)
        nms.nms_amplitudes(ctx, grid, amp)
        nms.nms_synchronize(ctx)
        assert nms.nms_get_info(ctx, "variant_used") == used
        if qt:
            assert nms.nms_get_info(ctx, "qt") == qt
        assert_amplitudes(amp.cpu().numpy(), A, wsum, f"W={W} variant={variant} qt={qt} precision={prec}")
    # the interpolating accurate kernel over the same ragged tiles (a finer |q| grid: its step phase must stay below 0.2 cycle)
    fine = ni.polar_grid(0.3 + 0.02 * np.arange(19), 37)
    qy, qz, th = oracle_mod.grid_points(fine)
    A, wsum = oracle_mod.amplitudes(pos, N, m, None, qy, qz, return_wsum=True)
    for key, value in (("variant", 2), ("qt", 16), ("precision", 2), ("interp", 2)):
        nms.nms_set_option(ctx, key, value)
    nms.nms_amplitudes(ctx, fine, amp)
    nms.nms_synchronize(ctx)
    assert nms.nms_get_info(ctx, "interp") == 1
    assert_amplitudes(amp.cpu().numpy(), A, wsum, f"W={W} interpolating kernel")


@pytest.mark.parametrize("variant,prec", [(0, 0), (1, 1), (1, 0)])
def test_list_grid_against_oracle(nms, ctx, oracle_mod, variant, prec):
    """A point-list detector with random non-zero q (MODE 2 kernel, 4 points per thread): amplitudes and all kinds."""
    import torch
    rng = np.random.Generator(np.random.Philox(606))
    W, n = 2500, 1003                                                 # 1003 points: ragged against 128 threads x 4 points
    pos = rng.uniform(-25, 25, size=(W, 3)).astype(np.float32)
    N = rng.uniform(0.5, 1.5, size=W).astype(np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    R = ni.rotation_alpha_beta(33.0, 71.0)
    grid = ni.list_grid(rng.uniform(-1.5, 1.5, size=n), rng.uniform(-1.5, 1.5, size=n))
    kinds = list(ni.ALL_KINDS)
    nms.nms_set_sample(ctx, _t(pos), _t(N), _t(m), R)
    nms.nms_set_option(ctx, "variant", variant)
    nms.nms_set_option(ctx, "precision", prec)
    amp = torch.empty((8, n), dtype=torch.float32, device="cuda")
    maps = torch.empty((len(kinds), n), dtype=torch.float32, device="cuda")
    nms.nms_amplitudes(ctx, grid, amp)
    nms.nms_response(ctx, kinds, maps)
    nms.nms_synchronize(ctx)
    assert nms.nms_get_info(ctx, "variant_used") == (1 if variant else 8)
    qy, qz, th = oracle_mod.grid_points(grid)
    A, wsum = oracle_mod.amplitudes(pos, N, m, R, qy, qz, return_wsum=True)
    M = oracle_mod.response(A, th, kinds)
    assert_amplitudes(amp.cpu().numpy(), A, wsum, "list grid")
    misses = [] if variant else None
    assert_cross_sections(maps.cpu().numpy(), M, kinds, "list grid", signed_misses=misses)
    report_signed_misses(misses)


@pytest.mark.parametrize("gtype", [0, 1])
def test_recurrence_far_from_the_origin(nms, ctx, oracle_mod, gtype):
    """A sample translated by ~1e3 nm: the float abscissae of the line deviate from the evaluated progression by up to
    one ulp(q), a phase of ulp(q) |r| ~ 1e-4 rad that the recurrence kernels correct at the tile centres; the exact
    phase reduction is indifferent to the offset (|t| ~ 500 cycles << 2^19)."""
    import torch
    rng = np.random.Generator(np.random.Philox(919))
    nx = 24
    g = (np.arange(nx) - (nx - 1) / 2.0)
    zz, yy, xx = np.meshgrid(g, g, g, indexing="ij")
    pos = (np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1) + np.array([300.0, 900.0, -700.0])).astype(np.float32)
    W = pos.shape[0]
    N = np.ones(W, dtype=np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    grid = ni.polar_grid(0.01 + np.arange(40) * (2.99 / 39), 48) if gtype == 0 else \
        ni.cartesian_grid(np.linspace(-2.0, 2.1, 40), np.linspace(-2.0, 2.0, 33))
    kinds = [KI[k] for k in ("NUC", "MAG", "UNPOL", "PROJ", "SF")]
    nms.nms_set_sample(ctx, _t(pos), _t(N), _t(m), None)
    qy, qz, th = oracle_mod.grid_points(grid)
    A, wsum = oracle_mod.amplitudes(pos, N, m, None, qy, qz, return_wsum=True)
    M = oracle_mod.response(A, th, kinds)
    amp = torch.empty((8, grid.n_q), dtype=torch.float32, device="cuda")
    maps = torch.empty((len(kinds), grid.n_q), dtype=torch.float32, device="cuda")
    for rec, prec in ((1, 1), (2, 1), (0, 2)):
        nms.nms_set_option(ctx, "variant", 2)
        nms.nms_set_option(ctx, "recurrence", rec)
        nms.nms_set_option(ctx, "precision", prec)
        nms.nms_amplitudes(ctx, grid, amp)
        nms.nms_response(ctx, kinds, maps)
        nms.nms_synchronize(ctx)
        assert nms.nms_get_info(ctx, "variant_used") == (3 if gtype == 0 else 5)
        assert_amplitudes(amp.cpu().numpy(), A, wsum, f"translated sample, recurrence {rec}")
        assert_cross_sections(maps.cpu().numpy(), M, kinds, f"translated sample, recurrence {rec}")


def test_phase_range_is_checked(nms, ctx):
    """The adder-rounding phase reduction holds for |t| < 2^19 cycles: beyond it the fp32 kernels refuse
    (NMS_E_UNSUPPORTED) instead of returning garbage; the exact kernel still runs."""
    import torch
    wl = ni.make_config("C1")
    pos = (wl.pos.astype(np.float64) + np.array([0.0, 3.0e6, 0.0])).astype(np.float32)   # q r / 2 pi = 1.4e6 cycles
    nms.nms_set_sample(ctx, _t(pos), _t(wl.N), _t(wl.m), None)
    out = torch.empty((1, wl.grid.n_q), dtype=torch.float32, device="cuda")
    nms.nms_set_option(ctx, "variant", 1)
    with pytest.raises(nms.NmsError) as e:
        nms.nms_compute(ctx, wl.grid, [0], out)
    assert e.value.status == nms.NMS_E_UNSUPPORTED
    nms.nms_set_option(ctx, "variant", 0)
    nms.nms_compute(ctx, wl.grid, [0], out)
    nms.nms_synchronize(ctx)
    assert nms.nms_get_info(ctx, "variant_used") == 8


def test_absent_channels(nms, ctx, oracle_mod):
    """N == NULL / m == NULL switch a channel off (L242): its amplitudes are exactly zero."""
    import torch
    wl = ni.make_config("C5", small=True)
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    for N, m in ((wl.N, None), (None, wl.m)):
        nms.nms_set_sample(ctx, _t(wl.pos), _t(N), _t(m), None)
        amp = torch.empty((8, wl.grid.n_q), dtype=torch.float32, device="cuda")
        nms.nms_amplitudes(ctx, wl.grid, amp)
        nms.nms_synchronize(ctx)
        A, wsum = oracle_mod.amplitudes(wl.pos, N, m, None, qy, qz, return_wsum=True)
        assert_amplitudes(amp.cpu().numpy(), A, wsum, "absent channel")


def test_general_polarization_and_scales(nms, ctx, oracle_mod):
    import torch
    wl = ni.make_config("C2")
    wl.P = np.array([0.3, -0.5, 0.8])
    _upload(nms, ctx, wl)
    nms.nms_set_scales(ctx, 2.5e-3, 0.7, 1.0 / 37.0)
    kinds = list(ni.ALL_KINDS)
    maps = torch.empty((len(kinds), wl.grid.n_q), dtype=torch.float32, device="cuda")
    nms.nms_compute(ctx, wl.grid, kinds, maps)
    nms.nms_synchronize(ctx)
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    A = oracle_mod.amplitudes(wl.pos, wl.N, wl.m, wl.R, qy, qz)
    M = oracle_mod.response(A, th, kinds, P=wl.P, sN=2.5e-3, sM=0.7, invV=1.0 / 37.0)
    assert_cross_sections(maps.cpu().numpy(), M, kinds, "general P")


def test_error_codes(nms, ctx):
    import torch
    wl = ni.make_config("C1")
    pos, N, m = _t(wl.pos), _t(wl.N), _t(wl.m)
    out = torch.empty((1, wl.grid.n_q), dtype=torch.float32, device="cuda")

    def status(fn, *a):
        with pytest.raises(nms.NmsError) as e:
            fn(*a)
        return e.value.status

    assert status(nms.nms_compute, ctx, wl.grid, [0], out) == nms.NMS_E_STATE            # no sample yet
    assert status(nms.nms_set_sample, ctx, pos, None, None, None) == nms.NMS_E_ARG        # no weights
    assert status(nms.nms_set_sample, ctx, pos, N, m, np.eye(3) * 1.01) == nms.NMS_E_ARG  # R not orthonormal
    nms.nms_set_sample(ctx, pos, N, m, None)
    assert status(nms.nms_response, ctx, [0], out) == nms.NMS_E_STATE                     # before nms_amplitudes
    assert status(nms.nms_compute, ctx, wl.grid, [99], out) == nms.NMS_E_ARG              # unknown kind
    assert status(nms.nms_form_factor_split, ctx, wl.grid, [0], out, out) == nms.NMS_E_STATE   # no particles
    assert status(nms.nms_set_particles, ctx, np.array([0, 5, 3, wl.W]), None) == nms.NMS_E_ARG
    assert status(nms.nms_set_particles, ctx, np.array([0, 5, wl.W - 1]), None) == nms.NMS_E_ARG
    assert status(nms.nms_set_polarization, ctx, [0, 0, 0]) == nms.NMS_E_ARG
    assert status(nms.nms_set_option, ctx, "nonsense", 1) == nms.NMS_E_ARG
    bad = ni.polar_grid(0.01 * 1.5 ** np.arange(8), 8)
    nms.nms_set_option(ctx, "variant", 2)
    assert status(nms.nms_compute, ctx, bad, [0], out[:, :64].contiguous()) == nms.NMS_E_UNSUPPORTED
    nms.nms_set_option(ctx, "variant", 0)
    nms.nms_compute(ctx, wl.grid, [0], out)                                             # context still usable
    nms.nms_synchronize(ctx)
    assert "" == nms.nms_last_error(ctx)


def test_run_host_matches_device_path(nms, ctx):
    import torch
    wl = ni.make_config("C2")
    kinds = wl.kinds
    nq, nb, nr = wl.grid.n_q, wl.n_bins, len(wl.r)
    out_maps = np.empty((len(kinds), nq), dtype=np.float32)
    out_I = np.empty((len(kinds), nb), dtype=np.float32)
    out_c = np.empty((len(kinds), nr), dtype=np.float32)
    out_p = np.empty_like(out_c)
    nms.nms_run_host(ctx, wl.pos, wl.N, wl.m, wl.R, wl.grid, kinds, out_maps, nb, wl.q_lo, wl.q_hi, out_I, wl.r, out_c, out_p)
    _upload(nms, ctx, wl)
    maps = torch.empty((len(kinds), nq), dtype=torch.float32, device="cuda")
    nms.nms_compute(ctx, wl.grid, kinds, maps)
    nms.nms_synchronize(ctx)
    assert np.array_equal(maps.cpu().numpy(), out_maps)
    I = torch.empty((len(kinds), nb), dtype=torch.float32, device="cuda")
    qb = torch.empty(nb, dtype=torch.float32, device="cuda")
    cnt = torch.empty(nb, dtype=torch.int32, device="cuda")
    c = torch.empty((len(kinds), nr), dtype=torch.float32, device="cuda")
    p = torch.empty_like(c)
    nms.nms_azimuthal_average(ctx, maps, len(kinds), nb, wl.q_lo, wl.q_hi, I, qb, cnt)
    nms.nms_correlation(ctx, I, qb, cnt, len(kinds), nb, _t(wl.r), c, p)
    nms.nms_synchronize(ctx)
    # same kernels on the same maps: the histogram adds with fp64 atomics whose order is not fixed (last-bit differences)
    np.testing.assert_allclose(out_I, I.cpu().numpy(), rtol=1e-6, atol=0)
    np.testing.assert_allclose(out_c, c.cpu().numpy(), rtol=1e-5, atol=1e-7 * np.abs(out_c).max())
    np.testing.assert_allclose(out_p, p.cpu().numpy(), rtol=1e-5, atol=1e-7 * np.abs(out_p).max())


def test_phasor_error_statistics(nms, ctx):
    """The two phasor routines of the amplitude kernels over 2^22 stratified phases against fp64 (nms_phasor_selftest):
    MUFU within the 2^-21.4 of the CUDA C Programming Guide plus the I2FP / FMUL roundings; the polynomial phasor at
    fp32 rounding level with every Fourier coefficient of its error function (the leakage of A(n q) into A(q)) below
    2e-9 -- the figures DESIGN.md section 7 quotes."""
    mufu = nms.nms_phasor_selftest(ctx, False, 22)
    poly = nms.nms_phasor_selftest(ctx, True, 22)
    assert max(mufu["max_cos"], mufu["max_sin"]) <= 6e-7
    assert max(poly["max_cos"], poly["max_sin"]) <= 1.2e-7
    assert max(poly["rms_cos"], poly["rms_sin"]) <= 3e-8
    assert all(v <= 2e-9 for n, v in poly["harmonics"].items())
    # the constant term of the MUFU error is the mean error of its cosine, 1.2758e-8 on B200 (it adds that times sum w to
    # every amplitude: DESIGN.md section 7 counts it among the causes of the signed-kind misses of the fp32 kernels)
    assert abs(mufu["mean_cos"] - 1.2758e-8) <= 3e-10 and abs(mufu["mean_minus_sin"]) <= 3e-10
    assert abs(poly["mean_cos"]) <= 1e-10


def test_pipe_rates_are_sane(nms, ctx):
    """The micro-benchmark behind the roofline denominators: 128 FP32 lanes and 16 MUFU lanes per clock and SM."""
    r = nms.nms_pipe_rates(ctx)
    assert 100.0 <= r["FFMA"] <= 135.0
    assert 100.0 <= r["FFMA2_BCAST"] <= 130.0              # lane-FMAs: a packed FFMA2 is two of them
    assert 12.0 <= r["MUFU_EX2"] <= 17.0
    assert r["PHASOR_POLY"] < r["FFMA"] / 8.0


@pytest.mark.parametrize("gtype,variant", [(0, 0), (1, 0), (2, 0), (0, 1), (1, 1), (0, 2), (1, 2)])
def test_batched_fields(nms, ctx, oracle_mod, gtype, variant):
    """f-3 (L254, L323, L391): B = 5 magnetisation fields (two passes: 3 + 2) on the geometry of the reduced C5, with a
    rotation: amplitudes of every field within 1e-5 sum|w| and all 13 kinds at the north_star criterion against the plain
    loop of the oracle; the nuclear planes are shared.  Polar, Cartesian and list detectors; variant 0: the library's
    choice (accurate variant: line recurrence over 8 points per thread on the equally spaced polar / Cartesian lines -- 19
    lines: ragged --; fast variant and list detector: direct), 1: the direct kernel forced, 2: the recurrence forced."""
    import torch
    wl = ni.make_config("C5", small=True)
    rng = np.random.Generator(np.random.Philox(808))
    B, W = 5, wl.W
    mb = np.stack([wl.m, np.roll(wl.m, 1, axis=1), -wl.m[:, ::-1], rng.normal(size=(W, 3)),
                   np.tile(np.array([0.0, 0.6, 0.8]), (W, 1))]).astype(np.float32)
    R = ni.rotation_alpha_beta(15.0, 35.0)
    grid = [wl.grid, ni.cartesian_grid(np.linspace(-1.4, 1.5, 19), np.linspace(-1.5, 1.5, 40)),
            ni.list_grid(rng.uniform(-2, 2, size=301), rng.uniform(-2, 2, size=301))][gtype]
    kinds = list(ni.ALL_KINDS)
    nms.nms_set_sample(ctx, _t(wl.pos), _t(wl.N), None, R)
    nq = grid.n_q
    maps = torch.empty((B, len(kinds), nq), dtype=torch.float32, device="cuda")
    amp = torch.empty((B, 8, nq), dtype=torch.float32, device="cuda")
    qy, qz, th = oracle_mod.grid_points(grid)
    A = oracle_mod.amplitudes_batch(wl.pos, wl.N, mb, R, qy, qz)
    misses = []
    for prec in (1, 0):                                     # fast (MUFU), then automatic = accurate (signed kinds asked for)
        nms.nms_set_option(ctx, "precision", prec)
        nms.nms_set_option(ctx, "variant", variant)
        nms.nms_compute_batch(ctx, grid, _t(mb), kinds, maps, amp)
        nms.nms_synchronize(ctx)
        assert (nms.nms_get_info(ctx, "poly_phasors") != 0) == (prec == 0)
        rec = gtype != 2 and (variant == 2 or (variant == 0 and prec == 0))
        assert nms.nms_get_info(ctx, "variant_used") == (17 if rec else 16)
        assert nms.nms_get_info(ctx, "qt") == (8 if rec else 4)
        assert nms.nms_get_info(ctx, "bases") == (1 if rec else 0)
        assert nms.nms_get_info(ctx, "three_term") == (1 if rec and prec == 1 else 0)
        a_h, m_h = amp.cpu().numpy(), maps.cpu().numpy()
        for b in range(B):
            _, wsum = oracle_mod.amplitudes(wl.pos, wl.N, mb[b], R, qy[:1], qz[:1], return_wsum=True)
            assert_amplitudes(a_h[b], A[b], wsum, f"field {b}")
            assert np.array_equal(a_h[b, 0:2], a_h[0, 0:2])                          # one nuclear amplitude for all fields
            M = oracle_mod.response(A[b], th, kinds)
            # the library's own choice (variant 0, automatic precision) is held to the criterion strictly; a forced
            # variant's misses of NM / CHI are reported
            strict = variant == 0 and prec == 0
            assert_cross_sections(m_h[b], M, kinds, f"field {b} precision {prec}", signed_misses=None if strict else misses)
    # the ordinary path on field 3 gives the same maps within the criterion
    nms.nms_set_sample(ctx, _t(wl.pos), _t(wl.N), _t(mb[3]), R)
    nms.nms_set_option(ctx, "variant", 1)
    nms.nms_set_option(ctx, "precision", 0)
    one = torch.empty((len(kinds), nq), dtype=torch.float32, device="cuda")
    nms.nms_compute(ctx, grid, kinds, one)
    nms.nms_synchronize(ctx)
    pos_k = [i for i, k in enumerate(kinds) if k not in SIGNED]
    np.testing.assert_allclose(one.cpu().numpy()[pos_k], m_h[3][pos_k], rtol=2e-3, atol=1e-6 * np.abs(m_h[3]).max())
    report_signed_misses(misses)


def test_batched_fields_errors(nms, ctx):
    import torch
    wl = ni.make_config("C1")
    out = torch.empty((1, 1, wl.grid.n_q), dtype=torch.float32, device="cuda")
    mb = _t(wl.m[None])
    with pytest.raises(nms.NmsError) as e:
        nms.nms_compute_batch(ctx, wl.grid, mb, [0], out, None)
    assert e.value.status == nms.NMS_E_STATE                       # no sample (geometry) yet
    nms.nms_set_sample(ctx, _t(wl.pos), _t(wl.N), None, None)
    with pytest.raises(nms.NmsError) as e:
        nms.nms_compute_batch(ctx, wl.grid, mb, [0], None, None)
    assert e.value.status == nms.NMS_E_ARG
    with pytest.raises(nms.NmsError) as e:
        nms.nms_compute_batch(ctx, wl.grid, mb, [77], out, None)
    assert e.value.status == nms.NMS_E_ARG
    nms.nms_compute_batch(ctx, wl.grid, mb, [0], out, None)
    nms.nms_synchronize(ctx)


@pytest.mark.parametrize("name,small,variant", [("C1", False, 0), ("C5", True, 1), ("C5", True, 2)])
def test_friedel_halving(nms, ctx, oracle_mod, name, small, variant):
    """f-4: with option "friedel" the sums run over the first half of every ring and the second half is the conjugate
    (A(-q) = A(q)^*, Eq. 42-43): amplitudes within 1e-5 sum|w| and the positive kinds at the north_star criterion
    against the oracle on the FULL grid (the float angles theta_j + pi are met within 2.4e-7 rad)."""
    import torch
    wl = ni.make_config(name, small=small)
    kinds = [KI[k] for k in ("NUC", "MAG", "UNPOL", "PROJ", "SF", "PP", "MM", "PM", "MP")]
    _upload(nms, ctx, wl)
    nms.nms_set_option(ctx, "variant", variant)
    nms.nms_set_option(ctx, "friedel", 1)
    nms.nms_set_option(ctx, "precision", 1)    # nms_amplitudes and nms_compute (positive kinds) would otherwise differ in variant
    nq = wl.grid.n_q
    amp = torch.empty((8, nq), dtype=torch.float32, device="cuda")
    maps = torch.empty((len(kinds), nq), dtype=torch.float32, device="cuda")
    maps2 = torch.empty_like(maps)
    nms.nms_amplitudes(ctx, wl.grid, amp)
    nms.nms_response(ctx, kinds, maps)
    nms.nms_compute(ctx, wl.grid, kinds, maps2)
    nms.nms_synchronize(ctx)
    assert torch.equal(maps, maps2)
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    A, wsum, M = _oracle_maps(oracle_mod, wl, qy, qz, th, kinds)
    a_h = amp.cpu().numpy()
    assert_amplitudes(a_h, A, wsum, "friedel")
    assert_cross_sections(maps.cpu().numpy(), M, kinds, "friedel")
    n0, n1 = wl.grid.n0, wl.grid.n1
    a3 = a_h.reshape(8, n0, n1)
    assert np.array_equal(a3[0::2, :, n1 // 2:], a3[0::2, :, :n1 // 2])          # the second half IS the conjugate
    assert np.array_equal(a3[1::2, :, n1 // 2:], -a3[1::2, :, :n1 // 2])
    # not admissible: odd number of angles, Cartesian detector, form-factor split
    out = torch.empty((1, 7 * 9), dtype=torch.float32, device="cuda")
    for bad in (ni.polar_grid(np.linspace(0.1, 1.0, 7), 9), ni.cartesian_grid(np.linspace(-1, 1, 7), np.linspace(-1, 1, 9))):
        with pytest.raises(nms.NmsError) as e:
            nms.nms_compute(ctx, bad, [0], out)
        assert e.value.status == nms.NMS_E_UNSUPPORTED
    nms.nms_set_option(ctx, "friedel", 0)
    nms.nms_compute(ctx, wl.grid, kinds, maps2)
    nms.nms_synchronize(ctx)
    assert_cross_sections(maps2.cpu().numpy(), M, kinds, "friedel off again")


def test_run_host_split_and_scan_match_device_path(nms, ctx):
    """The one-call host entry points of the per-particle split (C3's e2e arm) and of the rocking scan (C4's) give the
    maps of the device-resident call sequence bit for bit."""
    import torch
    w3 = ni.config_c3(K=7, n_q=21, n_theta=40, separate_centres=True)
    k3 = w3.kinds
    nq = w3.grid.n_q
    h_tot = np.empty((len(k3), nq), dtype=np.float32)
    h_form = np.empty_like(h_tot)
    nms.nms_run_host_split(ctx, w3.pos, w3.N, w3.m, w3.offsets, w3.centres, w3.R, w3.grid, k3, h_tot, h_form)
    _upload(nms, ctx, w3)
    tot = torch.empty((len(k3), nq), dtype=torch.float32, device="cuda")
    form = torch.empty_like(tot)
    nms.nms_form_factor_split(ctx, w3.grid, k3, tot, form)
    nms.nms_synchronize(ctx)
    assert np.array_equal(tot.cpu().numpy(), h_tot) and np.array_equal(form.cpu().numpy(), h_form)
    w4 = ni.make_config("C4", small=True)
    k4, nq4 = w4.kinds, w4.grid.n_q
    h_scan = np.empty((len(w4.rotations), len(k4), nq4), dtype=np.float32)
    nms.nms_run_host_scan(ctx, w4.pos, w4.N, w4.m, w4.rotations, w4.grid, k4, h_scan)
    nms.nms_set_sample(ctx, _t(w4.pos), _t(w4.N), _t(w4.m), w4.rotations[0])
    maps = torch.empty((len(k4), nq4), dtype=torch.float32, device="cuda")
    for i, R in enumerate(w4.rotations):
        nms.nms_set_rotation(ctx, R)
        nms.nms_compute(ctx, w4.grid, k4, maps)
        nms.nms_synchronize(ctx)
        assert np.array_equal(maps.cpu().numpy(), h_scan[i]), f"rotation {i}"
