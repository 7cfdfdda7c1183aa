"""GPU parity: the CUDA library (through its C-ABI binding) against the CPU oracle, element by
element, on the seeded workloads of BASELINE.json at sizes the oracle finishes in seconds that
still span several dispatch tiles and a ragged tail; plus sampled checks at full size.

Tolerances (BASELINE.json north_star): fp64 |flux_gpu - flux_oracle| <= 1e-9 absolute;
fp32 <= 2e-7 absolute.  Integer work (dispatch tiles, status words) is bit-exact.
"""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

TOL64 = 1e-9
TOL32 = 2e-7


@pytest.fixture(scope="module")
def rr():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (there is no CPU fallback)")
    import paper_2009_08500_b200 as m
    m.load()
    return m


def gpu_model(rr, wl, precision=0):
    model = rr.RoadRunner.from_config(wl.model, precision)
    model.set_data(wl.times, wl.lc_index, wl.passband_index, wl.supersampling, wl.exposure_time)
    return model


def gpu_flux(rr, wl, precision=0, reduction=0, want_status=False):
    model = gpu_model(rr, wl, precision)
    if reduction:
        rr.rr_set_reduction(model.ctx, reduction)
    model.build_ld_table(wl.ldp(model.mu))
    flux, status = model.evaluate(wl.pv, want_status=True)
    out = flux.cpu().numpy().astype(np.float64), status.cpu().numpy()
    model.close()
    return out if want_status else out[0]


def oracle_flux(wl):
    flux, status = oracle.evaluate_workload(wl, nthreads=0)
    return flux, status


SMALL = {  # config -> (npv, npt): several tiles per light curve and a ragged tail
    0: (None, None),
    1: (48, 5000),
    2: (12, 3000),
    3: (10, 6 * 2500),
    4: (40, 7001),
}


def small_workload(config):
    npv, npt = SMALL[config]
    return workloads.make_workload(config, npv=npv, npt=npt)


# ---- a0: geometry ------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", [dict(), dict(nzin=100, nzlimb=100, npb=4),
                                 dict(k0=0.01, k1=0.3), dict(nzin=7, nzlimb=5, ng=11, nk=3)])
def test_geometry_matches_oracle(rr, cfg):
    mc = workloads.ModelConfig(**cfg)
    om = oracle.OracleModel.from_config(mc)
    gm = rr.RoadRunner.from_config(mc)
    assert np.max(np.abs(gm.ze - om.ze)) <= 4e-16
    assert np.max(np.abs(gm.mu - om.mu)) <= 4e-16
    W = gm.weights()
    assert W.shape == om.W.shape
    assert np.max(np.abs(W - om.W)) <= 1e-11
    assert np.max(np.abs(W.sum(axis=2) - 1.0)) <= 1e-12
    gm.close()


# ---- kernel 1: LD table --------------------------------------------------------------------------------
@pytest.mark.parametrize("config,npv", [(0, None), (1, 300), (3, 37)])
def test_ld_table_matches_oracle(rr, config, npv):
    wl = workloads.make_workload(config, npv=npv, npt=600)
    om = oracle.OracleModel.from_config(wl.model)
    T_o, I_o = om.build_ld_table(wl.ldp(om.mu))
    gm = rr.RoadRunner.from_config(wl.model)
    gm.build_ld_table(wl.ldp(gm.mu))
    T_g, I_g = gm.table()
    assert T_g.shape == T_o.shape
    assert np.max(np.abs(T_g - T_o)) <= 1e-12
    assert np.max(np.abs(I_g / I_o - 1.0)) <= 1e-13
    gm.close()


def test_ld_table_istar_override(rr):
    wl = workloads.make_workload(1, npv=5, npt=300)
    gm = gpu_model(rr, wl)
    ldp = wl.ldp(gm.mu)
    given = np.linspace(2.0, 3.0, 5).reshape(5, 1)
    gm.build_ld_table(ldp, istar=given)
    _, I_g = gm.table()
    assert np.array_equal(I_g, given)
    flux_g = gm.evaluate(wl.pv).cpu().numpy()
    om = oracle.OracleModel.from_config(wl.model)
    om.build_ld_table(wl.ldp(om.mu), istar_override=given)
    flux_o, _ = om.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                            wl.exposure_time, wl.pv)
    assert np.max(np.abs(flux_g - flux_o)) <= TOL64
    gm.close()


# ---- kernels 2+3+4: flux, fp64 ---------------------------------------------------------------------------
@pytest.mark.parametrize("config", [0, 1, 2, 3, 4])
def test_flux_fp64_matches_oracle(rr, config):
    wl = small_workload(config)
    want, st_o = oracle_flux(wl)
    got, st_g = gpu_flux(rr, wl, want_status=True)
    assert got.shape == want.shape
    assert np.array_equal(st_g, st_o)
    err = np.abs(got - want)
    assert np.max(err) <= TOL64, (config, float(np.max(err)))
    # out of transit is 1 exactly on both sides
    assert np.array_equal(got == 1.0, want == 1.0) or np.max(err[(got == 1.0) != (want == 1.0)]) <= 1e-12
    assert (want < 1.0).sum() > 100 or config == 0


@pytest.mark.parametrize("config", [2, 3, 4])
def test_flux_fp32_matches_oracle(rr, config):
    wl = small_workload(config)
    want, _ = oracle_flux(wl)
    got = gpu_flux(rr, wl, precision=1)
    err = np.abs(got - want)
    assert np.max(err) <= TOL32, (config, float(np.max(err)))


@pytest.mark.parametrize("config", [2, 3])
@pytest.mark.parametrize("precision", [0, 1])
def test_reduction_layouts_agree(rr, config, precision):
    """Thread-per-exposure loop and lanes-over-sub-samples warp-shuffle sum: same flux."""
    wl = small_workload(config)
    want, _ = oracle_flux(wl)
    a = gpu_flux(rr, wl, precision, reduction=1)
    b = gpu_flux(rr, wl, precision, reduction=2)
    tol = TOL32 if precision else TOL64
    assert np.max(np.abs(a - want)) <= tol
    assert np.max(np.abs(b - want)) <= tol
    assert np.max(np.abs(a - b)) <= (1e-6 if precision else 1e-14)


@pytest.mark.parametrize("config,precision,shape", [
    (1, 0, None), (3, 0, None), (3, 1, None), (4, 0, None),
    (4, 0, (2500, 400)), (3, 0, (700, 6 * 60)), (3, 1, (700, 6 * 60))])   # >= 2048 rows: bucketed builder
def test_table_modes_agree(rr, config, precision, shape):
    """RR_TABLE_LAZY (rows for each pv's k at evaluate time; per-row builder
    below 2048 (pv, passband) rows, ik-bucketed builder above) and RR_TABLE_FULL (whole T, rows
    collapsed while staging): same flux to rounding, both within tolerance."""
    wl = small_workload(config) if shape is None else \
        workloads.make_workload(config, npv=shape[0], npt=shape[1])
    want, _ = oracle_flux(wl)
    out = {}
    for mode in (rr.RR_TABLE_LAZY, rr.RR_TABLE_FULL):
        gm = rr.RoadRunner.from_config(wl.model, precision)
        rr.rr_set_table_mode(gm.ctx, mode)
        gm.set_data(wl.times, wl.lc_index, wl.passband_index, wl.supersampling, wl.exposure_time)
        gm.build_ld_table(wl.ldp(gm.mu))
        out[mode] = gm.evaluate(wl.pv).cpu().numpy().astype(np.float64)
        gm.close()
    tol = TOL32 if precision else TOL64
    for got in out.values():
        assert np.max(np.abs(got - want)) <= tol
    assert np.max(np.abs(out[rr.RR_TABLE_LAZY] - out[rr.RR_TABLE_FULL])) <= (2e-7 if precision else 1e-14)


# ---- direct model on the device (NEXT-1) ---------------------------------------------------------------
def _direct_gpu(rr, wl, precision, pv=None):
    gm = rr.RoadRunner.from_config(wl.model, precision)
    rr.rr_set_table_mode(gm.ctx, rr.RR_TABLE_DIRECT)
    gm.set_data(wl.times, wl.lc_index, wl.passband_index, wl.supersampling, wl.exposure_time)
    gm.build_ld_table(wl.ldp(gm.mu))
    flux, status = gm.evaluate(wl.pv if pv is None else pv, want_status=True)
    rows = gm.rows().astype(np.float64)
    out = flux.cpu().numpy().astype(np.float64), status.cpu().numpy(), rows
    gm.close()
    return out


@pytest.mark.parametrize("config,precision", [(1, 0), (2, 0), (3, 0), (4, 0), (3, 1), (4, 1)])
def test_direct_model_matches_oracle(rr, config, precision):
    """RR_TABLE_DIRECT: rows = weights at the pv's own k contracted with the
    profile, then the same flux kernel; against the oracle's direct model."""
    wl = small_workload(config)
    om = oracle.OracleDirectModel.from_config(wl.model)
    rows_o, _ = om.rows(wl.ldp(om.mu), wl.pv)
    want, st_o = om.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                             wl.exposure_time, wl.pv, wl.ldp(om.mu), nthreads=0)
    got, st_g, rows_g = _direct_gpu(rr, wl, precision)
    assert np.array_equal(st_g, st_o)
    assert np.max(np.abs(rows_g - rows_o)) <= (2e-7 if precision else 1e-12)
    assert np.max(np.abs(got - want)) <= (TOL32 if precision else TOL64)
    assert (want < 1.0).sum() > 100


def test_direct_model_has_no_k_limits(rr):
    wl = workloads.make_workload(1, npv=6, npt=1500)
    pv = wl.pv.copy()
    pv[0, 0] = 0.45            # far above the table's k1: valid in the direct model
    pv[1, 0] = 0.004           # below k0: valid
    pv[2, 0] = -0.1            # k <= 0: invalid
    pv[3, 0] = np.nan
    om = oracle.OracleDirectModel.from_config(wl.model)
    want, st_o = om.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                             wl.exposure_time, pv, wl.ldp(om.mu))
    got, st_g, _ = _direct_gpu(rr, wl, 0, pv=pv)
    assert np.array_equal(st_g, st_o) and list(st_g[:4]) == [0, 0, 1, 16]
    assert np.array_equal(np.isnan(got), np.isnan(want))
    ok = ~np.isnan(want)
    assert np.max(np.abs(got[ok] - want[ok])) <= TOL64
    assert want[0].min() < 0.85


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_mean_k_weights_shortcut(rr, mode):
    """Transmission-spectroscopy shortcut (reading R13) with chromatic k, in the
    lazy, full-table and direct modes, against the oracle's statement of it."""
    mc = workloads.ModelConfig(npb=3, nkpb=3)
    rng = np.random.default_rng(8)
    base = workloads.make_workload(1, npv=9, npt=10).pv
    kk = np.clip(base[:, :1] * (1 + 0.05 * rng.uniform(-1, 1, (9, 3))), 0.021, 0.199)
    pv = np.concatenate([kk, base[:, 1:]], axis=1)
    times = np.tile(np.linspace(-0.15, 0.15, 700), 3)
    lc = np.repeat(np.arange(3, dtype=np.int32), 700)
    coeffs = rng.uniform(0.1, 0.4, (9, 3, 2))
    pbs, nss, ets = [0, 1, 2], [1, 1, 3], [0.0, 0.0, 0.01]
    if mode == 2:
        om = oracle.OracleDirectModel.from_config(mc)
        want, _ = om.evaluate(times, lc, pbs, nss, ets, pv,
                              workloads.sample_profile("quadratic", coeffs, om.mu),
                              mean_k_weights=True)
    else:
        om = oracle.OracleModel.from_config(mc)
        om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
        want, _ = om.evaluate(times, lc, pbs, nss, ets, pv, mean_k_weights=True)
        exact, _ = om.evaluate(times, lc, pbs, nss, ets, pv)
        assert np.max(np.abs(want - exact)) > 1e-7            # the shortcut is visible ...
    gm = rr.RoadRunner.from_config(mc)
    rr.rr_set_table_mode(gm.ctx, mode)
    rr.rr_set_mean_k_weights(gm.ctx, True)
    gm.set_data(times, lc, pbs, nss, ets)
    gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
    got = gm.evaluate(pv).cpu().numpy()
    assert np.max(np.abs(got - want)) <= TOL64                 # ... and the GPU takes the same one
    gm.close()


@pytest.mark.parametrize("mode,precision", [(2, 0), (0, 0), (2, 1)])
def test_small_planet_approximation(rr, mode, precision):
    """PAPER.md:184-186 (reading R14): pvs with k <= threshold take the profile at the planet's
    centre; the others are untouched.  Direct mode: every pv against the direct oracle with the
    same threshold.  Lazy mode: small pvs against that oracle, the rest against the table oracle."""
    wl = workloads.make_workload(4, npv=60, npt=3000)
    thr = 0.08
    small = wl.pv[:, 0] <= thr
    assert 5 < small.sum() < 55
    od = oracle.OracleDirectModel.from_config(wl.model)
    want_d, _ = od.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                            wl.exposure_time, wl.pv, wl.ldp(od.mu), nthreads=0, small_planet_k=thr)
    want_t, _ = oracle_flux(wl)
    gm = rr.RoadRunner.from_config(wl.model, precision)
    rr.rr_set_table_mode(gm.ctx, mode)
    rr.rr_set_small_planet(gm.ctx, thr)
    gm.set_data(wl.times, wl.lc_index, wl.passband_index, wl.supersampling, wl.exposure_time)
    gm.build_ld_table(wl.ldp(gm.mu))
    got = gm.evaluate(wl.pv).cpu().numpy().astype(np.float64)
    tol = TOL32 if precision else TOL64
    assert np.max(np.abs(got[small] - want_d[small])) <= tol
    ref = want_d if mode == 2 else want_t
    assert np.max(np.abs(got[~small] - ref[~small])) <= tol
    assert np.max(np.abs(want_d[small] - want_t[small])) > 1e-7     # the approximation is visible
    if mode == 0:                                                   # a full table cannot do it
        rr.rr_set_table_mode(gm.ctx, rr.RR_TABLE_FULL)
        gm.build_ld_table(wl.ldp(gm.mu))
        with pytest.raises(rr.RoadRunnerError) as e:
            gm.evaluate(wl.pv)
        assert e.value.code == -5
    gm.close()


# ---- seeded random set-ups: odd resolutions, ragged light curves, every mode -------------------------------
@pytest.mark.parametrize("seed", range(8))
def test_random_setups_match_oracle(rr, seed):
    """Model resolutions that are not multiples of anything (nz, ng, nk), light curves of ragged
    lengths in random order with random ns / exposure times / passbands, chromatic or achromatic k,
    circular and eccentric pvs mixed: lazy, full and direct modes against their oracles."""
    rng = np.random.default_rng(1000 + seed)
    npb = int(rng.integers(1, 4))
    nkpb = npb if rng.random() < 0.5 else 1
    mc = workloads.ModelConfig(nzin=int(rng.integers(3, 40)), nzlimb=int(rng.integers(3, 60)),
                               zcut=float(rng.uniform(0.4, 0.9)), ng=int(rng.integers(5, 140)),
                               nk=int(rng.integers(2, 30)), k0=0.03, k1=0.25, npb=npb, nkpb=nkpb)
    npv = int(rng.integers(1, 20))
    base = workloads.make_workload(4, npv=npv, npt=10).pv
    kk = rng.uniform(0.035, 0.24, (npv, nkpb))
    pv = np.concatenate([kk, base[:, 1:]], axis=1)
    pv[:, nkpb + 2] = np.maximum(pv[:, nkpb + 2], (1.3 + kk.max(axis=1)) / (1 - pv[:, nkpb + 4]))
    nlc = int(rng.integers(1, 6))
    lens = rng.integers(1, 1400, nlc)
    order = rng.permutation(nlc)
    times = np.concatenate([rng.uniform(-0.4, 0.4, lens[l]) for l in order])
    lc = np.concatenate([np.full(lens[l], l, np.int32) for l in order])
    pbs = rng.integers(0, npb, nlc)
    nss = rng.choice([1, 2, 3, 7, 16, 33], nlc)
    ets = rng.uniform(0.0, 0.05, nlc)
    coeffs = np.stack([rng.uniform(0.1, 0.6, (npv, npb)), rng.uniform(0.0, 0.3, (npv, npb))], -1)
    om = oracle.OracleModel.from_config(mc)
    om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
    want_t, st_t = om.evaluate(times, lc, pbs, nss, ets, pv)
    od = oracle.OracleDirectModel.from_config(mc)
    want_d, _ = od.evaluate(times, lc, pbs, nss, ets, pv,
                            workloads.sample_profile("quadratic", coeffs, od.mu))
    for mode, want in ((0, want_t), (1, want_t), (2, want_d)):
        for precision in (0, 1):
            gm = rr.RoadRunner.from_config(mc, precision)
            rr.rr_set_table_mode(gm.ctx, mode)
            gm.set_data(times, lc, pbs, nss, ets)
            gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
            got, st = gm.evaluate(pv, want_status=True)
            got = got.cpu().numpy().astype(np.float64)
            assert np.array_equal(st.cpu().numpy(), st_t)
            err = float(np.max(np.abs(got - want)))
            assert err <= (TOL32 if precision else TOL64), (seed, mode, precision, err)
            gm.close()


def test_bucketed_row_builder_with_chromatic_k(rr):
    """>= 2048 (pv, passband) rows with one k per passband: the ik-bucketed lazy builder must bucket
    every row by ITS passband's k.  Rows against the direct statement (1-ak) T[ik] + ak T[ik+1] from
    the oracle's table; flux against the oracle."""
    mc = workloads.ModelConfig(npb=3, nkpb=3)
    rng = np.random.default_rng(21)
    npv = 700
    base = workloads.make_workload(1, npv=npv, npt=10).pv
    kk = rng.uniform(0.021, 0.199, (npv, 3))
    pv = np.concatenate([kk, base[:, 1:]], axis=1)
    times = np.tile(np.linspace(-0.2, 0.2, 60), 3)
    lc = np.repeat(np.arange(3, dtype=np.int32), 60)
    coeffs = rng.uniform(0.1, 0.4, (npv, 3, 2))
    om = oracle.OracleModel.from_config(mc)
    T, _ = om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
    want, _ = om.evaluate(times, lc, [0, 1, 2], [1, 2, 1], [0.0, 0.01, 0.0], pv, nthreads=0)
    gm = rr.RoadRunner.from_config(mc)
    gm.set_data(times, lc, [0, 1, 2], [1, 2, 1], [0.0, 0.01, 0.0])
    gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
    got = gm.evaluate(pv).cpu().numpy()
    rows = gm.rows()
    dk = (mc.k1 - mc.k0) / (mc.nk - 1)
    x = (kk - mc.k0) / dk
    ik = np.minimum(np.floor(x).astype(int), mc.nk - 2)
    ak = x - ik
    v, b = np.meshgrid(np.arange(npv), np.arange(3), indexing="ij")
    rows_o = (1 - ak)[..., None] * T[v, b, ik] + ak[..., None] * T[v, b, ik + 1]
    assert np.max(np.abs(rows - rows_o)) <= 1e-13
    assert np.max(np.abs(got - want)) <= TOL64
    gm.close()


def test_maximum_resolutions(rr):
    """ng and nz near the library's limits: the flux and direct-row kernels opt in to > 48 kB of
    dynamic shared memory (ng = 5000 staged nodes; direct rows with nz = 1500 edges)."""
    mc = workloads.ModelConfig(nzin=700, nzlimb=800, ng=5000, nk=3, k0=0.05, k1=0.15)
    wl = workloads.make_workload(1, npv=3, npt=900)
    wl.pv[:, 0] = [0.06, 0.1, 0.149]
    coeffs = wl.ld_coeffs
    om = oracle.OracleModel.from_config(mc)
    om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
    want_t, _ = om.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                            wl.exposure_time, wl.pv)
    od = oracle.OracleDirectModel.from_config(mc)
    want_d, _ = od.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                            wl.exposure_time, wl.pv, workloads.sample_profile("quadratic", coeffs, od.mu))
    for mode, want in ((0, want_t), (2, want_d)):
        gm = rr.RoadRunner.from_config(mc)
        rr.rr_set_table_mode(gm.ctx, mode)
        gm.set_data(wl.times, wl.lc_index, wl.passband_index, wl.supersampling, wl.exposure_time)
        gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
        got = gm.evaluate(wl.pv).cpu().numpy()
        assert np.max(np.abs(got - want)) <= TOL64
        gm.close()
    assert (want_t < 1).sum() > 100


# ---- mixed precision (NEXT-4) ------------------------------------------------------------
@pytest.mark.parametrize("config", [2, 3, 4])
def test_mixed_precision_scheme(rr, config):
    """RR_MIXED: z and Ip*Ap in fp32, their average over the sub-samples and 1 - avg/Istar in fp64,
    fp64 flux out (the scheme PAPER.md:293 proposes).  Error against the fp64 oracle: measured, and
    clearly below the fp32 mode's (whose stored flux alone is rounded to 6e-8 near 1)."""
    wl = small_workload(config)
    want, st_o = oracle_flux(wl)
    got32 = gpu_flux(rr, wl, precision=1)
    gm = gpu_model(rr, wl, precision=rr.RR_MIXED)
    gm.build_ld_table(wl.ldp(gm.mu))
    flux, status = gm.evaluate(wl.pv, want_status=True)
    assert flux.dtype == __import__("torch").float64
    gotm = flux.cpu().numpy()
    assert np.array_equal(status.cpu().numpy(), st_o)
    em, e32 = np.max(np.abs(gotm - want)), np.max(np.abs(got32 - want))
    assert em <= 2e-8 and em < 0.6 * e32, (config, em, e32)
    assert np.array_equal(gotm == 1.0, want == 1.0)
    status_h = np.empty(wl.npv, np.int32)
    host = gm.evaluate_host(wl.ldp(gm.mu), wl.pv, status=status_h)
    assert host.dtype == np.float64 and np.array_equal(host, gotm)
    gm.close()


# ---- named laws on the device (NEXT-4) ------------------------------------------------------------------
LAWS = [("uniform", None), ("linear", [(0.2, 0.8)]), ("quadratic", [(0.1, 0.6), (0.0, 0.3)]),
        ("quadratic-tri", [(0.1, 0.8), (0.1, 0.5)]), ("general", [(0.1, 0.4), (0.0, 0.2), (-0.1, 0.1)]),
        ("nonlinear", [(0.1, 0.5), (-0.2, 0.2), (0.1, 0.4), (-0.2, 0.1)]),
        ("logarithmic", [(0.3, 0.7), (0.0, 0.3)]), ("exponential", [(0.3, 0.6), (0.0, 0.02)]),
        ("power-2", [(0.3, 0.9), (0.3, 1.2)]), ("power-2-pm", [(0.6, 0.8), (0.35, 0.55)])]


@pytest.mark.parametrize("name,ranges", LAWS)
@pytest.mark.parametrize("precision", [0, 1])
def test_named_laws_on_device(rr, name, ranges, precision):
    """rr_build_ld_table_law: the law evaluated on the device at the library's mu grid with its
    closed-form Istar, against the test harness's statement of the same law
    (oracle/truth.py, disc integrals pinned to quadrature) fed through the table oracle."""
    from oracle import truth
    mc = workloads.ModelConfig(npb=2)
    base = workloads.make_workload(1, npv=7, npt=10)
    rng = np.random.default_rng(12)
    ldc = None if ranges is None else np.stack(
        [rng.uniform(lo, hi, (7, 2)) for lo, hi in ranges], axis=-1)
    times = np.tile(np.linspace(-0.2, 0.2, 800), 2)
    lc = np.repeat(np.arange(2, dtype=np.int32), 800)
    om = oracle.OracleModel.from_config(mc)
    ldp = np.empty((7, 2, om.nz))
    ist = np.empty((7, 2))
    for v in range(7):
        for b in range(2):
            f, i0 = truth.law(name, [] if ldc is None else ldc[v, b])
            ldp[v, b] = f(om.mu)
            ist[v, b] = np.nan if i0 is None else i0
    closed = not np.isnan(ist).any()
    om.build_ld_table(ldp, istar_override=ist if closed else None)
    want, _ = om.evaluate(times, lc, [0, 1], [1, 2], [0.0, 0.01], base.pv)
    gm = rr.RoadRunner.from_config(mc, precision)
    gm.set_data(times, lc, [0, 1], [1, 2], [0.0, 0.01])
    gm.npv = 7
    gm.build_ld_table_law(name, ldc)
    got = gm.evaluate(base.pv).cpu().numpy().astype(np.float64)
    I_g = gm.profile_and_istar().astype(np.float64)
    assert np.max(np.abs(I_g / om.istar - 1.0)) <= (3e-7 if precision else 1e-13)
    assert np.max(np.abs(got - want)) <= (TOL32 if precision else TOL64)
    assert (want < 1).sum() > 200
    gm.close()


def test_named_law_argument_errors(rr):
    import torch
    gm = rr.RoadRunner()
    ldc = torch.zeros((3, 1, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_build_ld_table_law(gm.ctx, "quadratic", ldc, 3)      # needs 2 coefficients
    assert e.value.code == -3
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_build_ld_table_law(gm.ctx, 17, ldc, 3)
    assert e.value.code == -2
    gm.close()


def test_kernel_timing_counts_calls(rr):
    wl = small_workload(1)
    gm = gpu_model(rr, wl)
    gm.build_ld_table(wl.ldp(gm.mu))
    rr.rr_enable_kernel_timing(gm.ctx, True)
    for _ in range(3):
        gm.evaluate(wl.pv)
    t = rr.rr_get_kernel_times(gm.ctx)
    assert t["calls"] == 3 and t["flux_ms"] > 0 and t["rows_ms"] > 0
    assert rr.rr_get_kernel_times(gm.ctx)["calls"] == 0
    gm.close()


# ---- kernel 2 alone ------------------------------------------------------------------------------------
@pytest.mark.parametrize("config", [1, 3, 4])
def test_orbit_z_matches_oracle(rr, config):
    wl = workloads.make_workload(config, npv=24, npt=6 * 200 if config == 3 else 1500)
    _, _, z_o = oracle.evaluate_workload(wl, want_z=True)
    gm = gpu_model(rr, wl)
    assert rr.rr_num_subsamples(gm.ctx) == z_o.shape[1]
    z_g = gm.orbit_z(wl.pv).cpu().numpy()
    assert np.max(np.abs(z_g - z_o)) <= 1e-11 * max(1.0, float(np.max(np.abs(z_o))))
    z32 = gm.orbit_z(wl.pv, fp32_math=True).cpu().numpy()
    # fp32 orbit arithmetic (diagnostic of the RR_FP32 flux kernel's kernel-2 part; the binding fp32
    # bar is the 2e-7 flux tolerance above).  The residual of Kepler's equation is formed in fp32,
    # so d carries ~3 eps |dM| / (1 - e cos E): a few 1e-6 in z at e = 0.7.
    near = np.abs(z_o) < 1.5         # the part of the orbit that matters
    assert np.max(np.abs(np.abs(z32[near]) - np.abs(z_o[near]))) <= 5e-6
    gm.close()


def test_orbit_high_eccentricity_full_phase(rr):
    """Solver robustness away from the transit window: e up to 0.95, every phase."""
    rng = np.random.default_rng(7)
    n = 64
    pv = np.empty((n, 7))
    pv[:, 0] = 0.1
    pv[:, 1] = rng.uniform(-0.5, 0.5, n)
    pv[:, 2] = rng.uniform(1.0, 5.0, n)
    pv[:, 3] = rng.uniform(30.0, 60.0, n)
    pv[:, 4] = rng.uniform(1.3, 1.6, n)
    pv[:, 5] = np.linspace(0.0, 0.95, n)
    pv[:, 6] = rng.uniform(0, 2 * np.pi, n)
    times = np.linspace(-6.0, 6.0, 2400)
    mc = workloads.ModelConfig()
    gm = rr.RoadRunner.from_config(mc)
    gm.set_data(times, np.zeros(times.size, np.int32), [0], [1], [0.0])
    z_g = gm.orbit_z(pv).cpu().numpy()
    z_o = np.array([[(lambda zf: zf[0] if zf[1] else -zf[0])(oracle.separation(t, *row[1:]))
                     for t in times] for row in pv])
    assert np.max(np.abs(z_g - z_o) / np.maximum(1.0, np.abs(z_o))) <= 1e-11
    gm.close()


# ---- kernel 4: dispatch -----------------------------------------------------------------------------------
TILE_UNIT, TILE_SPAN = 1024, 0.1


def expected_tiles(lc_index, supersampling, times):
    """Runs of equal lc_index cut into tiles: at most TILE_UNIT*R exposures, R = clamp((8+ns//2)//ns,
    1, 8), and no longer than TILE_SPAN days at the run's mean cadence, in multiples of 128 (>= 128);
    the two floating-point roundings are those of rr_k4_run_tile_len."""
    tiles = []
    n = len(lc_index)
    b = 0
    while b < n:
        e = b
        while e < n and lc_index[e] == lc_index[b]:
            e += 1
        ns = int(supersampling[lc_index[b]])
        max_len = TILE_UNIT * max(1, min(8, (8 + ns // 2) // ns))
        length = max_len
        if e - b >= 2:
            with np.errstate(divide="ignore", invalid="ignore"):
                span = np.abs(np.float64(times[e - 1]) - np.float64(times[b]))
                cnt = np.float64(e - b - 1) * (np.float64(TILE_SPAN) / span)
            if cnt < max_len:
                length = min(max(128, (int(cnt) + 127) // 128 * 128), max_len)
        for s in range(b, e, length):
            tiles.append((s, min(length, e - s), int(lc_index[b])))
        b = e
    return tiles


@pytest.mark.parametrize("case", ["config3", "interleaved", "single", "paper", "sparse"])
def test_dispatch_tiles(rr, case):
    rng = np.random.default_rng(11)
    if case == "config3":
        wl = workloads.make_workload(3, npv=1, npt=6 * 2500)
        times, lc, pb, ns, et = wl.times, wl.lc_index, wl.passband_index, wl.supersampling, \
            wl.exposure_time
        npb = 4
    elif case == "interleaved":
        lc = rng.integers(0, 3, 5000).astype(np.int32)
        lc[1000:3500] = 2
        times = rng.uniform(-1, 1, lc.size)
        pb, ns, et, npb = [0, 1, 0], [1, 7, 30], [0.0, 0.01, 0.02], 2
    elif case == "sparse":                     # 2-minute cadence over 28 d: 128-exposure tiles
        lc = np.repeat(np.array([0, 1], np.int32), [20000, 777])
        times = np.concatenate([np.arange(20000) * (2.0 / 1440.0), 5.0 + np.arange(777) * 0.02])
        pb, ns, et, npb = [0, 0], [3, 10], [2.0 / 1440.0, 0.02], 1
    elif case == "single":
        lc = np.zeros(1, np.int32)
        times = np.array([0.25])
        pb, ns, et, npb = [0], [3], [0.01], 1
    else:
        d = workloads.paper_dummy_example()
        times, lc, pb = d["times"], d["lc_index"], d["passband_index"]
        ns, et, npb = [1, 2, 3], [0.0, 0.1, 0.2], 2
    gm = rr.RoadRunner(npb=npb)
    gm.set_data(times, lc, pb, ns, et)
    got = rr.rr_get_tiles(gm.ctx)
    want = expected_tiles(lc, ns, times)
    assert rr.rr_num_tiles(gm.ctx) == len(want)
    assert [(int(s), int(c), int(l)) for s, c, l in zip(got["start"], got["count"], got["lc"])] \
        == want
    for (s, c, _), lo, hi in zip(want, got["tmin"], got["tmax"]):
        assert lo == times[s:s + c].min() and hi == times[s:s + c].max()
    assert rr.rr_num_subsamples(gm.ctx) == int(np.asarray(ns)[lc].sum())
    gm.close()


def test_paper_dummy_example_indexing(rr):
    """points 0,1,5 use passband 0's table, points 2,3,4 passband 1's."""
    d = workloads.paper_dummy_example()
    times = d["times"] * 0.02 - 0.05
    mc = workloads.ModelConfig(npb=2)
    pv = np.array([[0.1, 0.0, 3.0, 8.0, np.deg2rad(88.0), 0.0, 0.0],
                   [0.15, 0.01, 2.0, 6.0, np.deg2rad(87.0), 0.2, 1.0]])
    coeffs = np.array([[[0.4, 0.2], [0.7, 0.1]], [[0.3, 0.3], [0.1, 0.05]]])
    ns, et = [1, 3, 2], [0.0, 0.01, 0.02]
    om = oracle.OracleModel.from_config(mc)
    om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
    want, _ = om.evaluate(times, d["lc_index"], d["passband_index"], ns, et, pv)
    gm = rr.RoadRunner.from_config(mc)
    gm.set_data(times, d["lc_index"], d["passband_index"], ns, et)
    gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
    got = gm.evaluate(pv).cpu().numpy()
    assert np.max(np.abs(got - want)) <= TOL64
    assert (want < 1).sum() >= 10
    gm.close()


def test_unsorted_times_and_out_of_order_light_curves(rr):
    wl = workloads.make_workload(3, npv=6, npt=6 * 700)
    rng = np.random.default_rng(5)
    perm = rng.permutation(wl.npt)
    wl = wl.subset_times(perm)
    want, _ = oracle_flux(wl)
    got = gpu_flux(rr, wl)
    assert np.max(np.abs(got - want)) <= TOL64


# ---- edge cases ---------------------------------------------------------------------------------------------
def test_invalid_parameter_vectors_give_nan_rows(rr):
    wl = workloads.make_workload(4, npv=12, npt=900)
    pv = wl.pv.copy()
    pv[1, 0] = 0.5          # k above k1
    pv[2, 5] = 1.0          # e = 1
    pv[3, 3] = -1.0         # a <= 0
    pv[4, 2] = 0.0          # p <= 0
    pv[5, 1] = np.nan
    pv[6, 0] = 0.001        # k below k0
    pv[7, 5] = -0.1
    wl.pv = pv
    want, st_o = oracle_flux(wl)
    got, st_g = gpu_flux(rr, wl, want_status=True)
    assert np.array_equal(st_g, st_o)
    assert list(st_g[:8]) == [0, 1, 2, 4, 8, 16, 1, 2]
    assert np.array_equal(np.isnan(got), np.isnan(want))
    ok = ~np.isnan(want)
    assert np.max(np.abs(got[ok] - want[ok])) <= TOL64


def test_grazing_wide_window_and_secondary_eclipse(rr):
    """a(1-e) barely above 1+k (window = whole orbit), periods short enough that the time span
    reaches the secondary-eclipse phase (flux must be 1 there), k at both table edges."""
    mc = workloads.ModelConfig()
    pv = np.array([
        [0.2, 0.0, 1.0, 1.25, np.deg2rad(80.0), 0.0, 0.0],
        [0.02, 0.1, 0.7, 2.0, np.deg2rad(89.0), 0.45, 4.0],
        [0.2, -0.2, 0.9, 3.0, np.deg2rad(75.0), 0.55, 1.0],
        [0.11, 0.0, 1.3, 1.6, np.deg2rad(60.0), 0.1, 2.5],
        [0.05, 0.3, 5.0, 12.0, np.deg2rad(90.0), 0.0, 0.0],
    ])
    times = np.linspace(-1.0, 1.0, 4001)
    coeffs = np.tile(np.array([[[0.5, 0.1]]]), (pv.shape[0], 1, 1))
    for ns, tau in ((1, 0.0), (4, 0.03)):
        om = oracle.OracleModel.from_config(mc)
        om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
        want, _ = om.evaluate(times, np.zeros(times.size, np.int32), [0], [ns], [tau], pv)
        gm = rr.RoadRunner.from_config(mc)
        gm.set_data(times, np.zeros(times.size, np.int32), [0], [ns], [tau])
        gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
        got = gm.evaluate(pv).cpu().numpy()
        assert np.max(np.abs(got - want)) <= TOL64
        gm.close()


@pytest.mark.parametrize("precision", [0, 1])
def test_long_exposures_many_subsamples_and_distant_epochs(rr, precision):
    """Degenerate corners of the supersampling path: an exposure longer than half the period (the
    phase of its sub-samples wraps), ns = 1000 sub-samples in one exposure (both reduction layouts
    through RR_REDUCE_AUTO), and epochs hundreds of periods away from t0."""
    mc = workloads.ModelConfig()
    pv = np.array([
        [0.1, 0.0, 1.0, 6.0, np.deg2rad(88.0), 0.0, 0.0],
        [0.15, 0.05, 1.3, 5.0, np.deg2rad(86.0), 0.4, 2.0],
        [0.05, -0.1, 2.7, 9.0, np.deg2rad(89.0), 0.2, 5.0],
        [0.2, 0.2, 0.8, 3.0, np.deg2rad(80.0), 0.6, 0.3],
    ])
    coeffs = np.tile(np.array([[[0.4, 0.25]]]), (pv.shape[0], 1, 1))
    t_a = np.linspace(-0.6, 0.6, 300)                     # lc 0: exposure 0.7 d > p/2 for pv 0, 3
    t_b = np.linspace(-0.05, 0.05, 7)                     # lc 1: ns = 1000
    t_c = 300.0 * 1.3 + np.linspace(-0.1, 0.1, 400)       # lc 2: 300 periods of pv 1 later
    times = np.concatenate([t_a, t_b, t_c])
    lc = np.concatenate([np.zeros(300), np.ones(7), np.full(400, 2)]).astype(np.int32)
    pbs, nss, ets = [0, 0, 0], [9, 1000, 2], [0.7, 0.02, 0.001]
    om = oracle.OracleModel.from_config(mc)
    om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
    want, _ = om.evaluate(times, lc, pbs, nss, ets, pv, nthreads=0)
    gm = rr.RoadRunner.from_config(mc, precision)
    gm.set_data(times, lc, pbs, nss, ets)
    gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
    got = gm.evaluate(pv).cpu().numpy().astype(np.float64)
    # 300 periods away the phase itself carries 300 * eps of rounding: ~1e-13 in z, no more
    assert np.max(np.abs(got - want)) <= (TOL32 if precision else TOL64)
    assert (want[:, :300] < 1).sum() > 200 and (want[:, 307:] < 1).sum() > 50
    gm.close()


@pytest.mark.parametrize("precision", [0, 1, 2])
def test_non_finite_times(rr, precision):
    """Reading R15: NaN / infinite times give NaN flux for those exposures in every layout
    (thread per exposure, lanes over sub-samples); everything else matches the oracle."""
    wl = workloads.make_workload(3, npv=5, npt=6 * 300)
    rng = np.random.default_rng(9)
    bad = rng.choice(wl.npt, 25, replace=False)
    wl.times[bad] = rng.choice([np.nan, np.inf, -np.inf], 25)
    want, _ = oracle_flux(wl)
    for reduction in (1, 2):
        got = gpu_flux(rr, wl, precision=precision, reduction=reduction)
        assert np.array_equal(np.isnan(got), np.isnan(want)) and np.isnan(want).sum() == 25 * 5
        ok = ~np.isnan(want)
        assert np.max(np.abs(got[ok] - want[ok])) <= {0: TOL64, 1: TOL32, 2: 2e-8}[precision]


def test_uniform_disk_closed_form(rr):
    """ldp = 1: flux = 1 - a(z,k)/pi straight from the CUDA path."""
    wl = workloads.make_workload(1, npv=8, npt=2000)
    wl.ld_kind = "uniform"
    gm = gpu_model(rr, wl)
    gm.build_ld_table(wl.ldp(gm.mu))
    flux = gm.evaluate(wl.pv).cpu().numpy()
    z = np.abs(gm.orbit_z(wl.pv).cpu().numpy())
    for v in range(wl.npv):
        k = wl.pv[v, 0]
        want = np.array([1.0 - oracle.lens_area(1.0, k, zz) / np.pi for zz in z[v]])
        assert np.max(np.abs(flux[v] - want)) <= 1e-13
    gm.close()


def test_chromatic_k(rr):
    """k per passband: pv rows carry npb radius ratios."""
    mc = workloads.ModelConfig(npb=2, nkpb=2)
    rng = np.random.default_rng(3)
    base = workloads.make_workload(1, npv=6, npt=10)
    pv = np.concatenate([base.pv[:, :1], base.pv[:, :1] * rng.uniform(0.9, 1.1, (6, 1)),
                         base.pv[:, 1:]], axis=1)
    pv[:, :2] = np.clip(pv[:, :2], 0.02, 0.2)
    times = np.tile(np.linspace(-0.2, 0.2, 900), 2)
    lc = np.repeat(np.arange(2, dtype=np.int32), 900)
    coeffs = rng.uniform(0.1, 0.4, (6, 2, 2))
    om = oracle.OracleModel.from_config(mc)
    om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
    want, _ = om.evaluate(times, lc, [0, 1], [1, 3], [0.0, 0.01], pv)
    gm = rr.RoadRunner.from_config(mc)
    gm.set_data(times, lc, [0, 1], [1, 3], [0.0, 0.01])
    gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
    got = gm.evaluate(pv).cpu().numpy()
    assert np.max(np.abs(got - want)) <= TOL64
    gm.close()


def test_paper_call_shapes(rr):
    """scalar parameters -> flux (npt,); arrays of npv -> (npv, npt); same values
    as the pv-matrix call."""
    wl = workloads.make_workload(3, npv=5, npt=6 * 40)
    gm = gpu_model(rr, wl)
    gm.build_ld_table(np.repeat(wl.ldp(gm.mu)[:1], 5, axis=0))
    pv = wl.pv
    ref = gm.evaluate(pv).cpu().numpy()
    many = gm.evaluate_ps(pv[:, 0], pv[:, 1], pv[:, 2], pv[:, 3], pv[:, 4], pv[:, 5], pv[:, 6])
    assert tuple(many.shape) == (5, wl.npt) and np.array_equal(many.cpu().numpy(), ref)
    gm.build_ld_table(wl.ldp(gm.mu)[:1])
    one = gm.evaluate_ps(*[float(x) for x in pv[0]])
    assert tuple(one.shape) == (wl.npt,) and np.array_equal(one.cpu().numpy(), ref[0])
    circ = gm.evaluate_ps(0.1, 0.0, 3.0, 8.0, 1.53)               # e, w default to 0
    assert tuple(circ.shape) == (wl.npt,) and float(circ.min()) < 1.0
    gm.close()


def test_argument_errors(rr):
    import torch
    gm = rr.RoadRunner()
    pv = torch.zeros((2, 7), dtype=torch.float64, device="cuda")
    flux = torch.zeros((2, 10), dtype=torch.float64, device="cuda")
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_evaluate(gm.ctx, pv, flux)               # no data, no table
    assert e.value.code == -5
    t = torch.linspace(-0.1, 0.1, 10, dtype=torch.float64, device="cuda")
    lc = torch.zeros(10, dtype=torch.int32, device="cuda")
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_set_data(gm.ctx, t, lc, [1], [1], [0.0])  # passband out of range
    assert e.value.code == -4
    bad = lc.clone()
    bad[3] = 2
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_set_data(gm.ctx, t, bad, [0], [1], [0.0])  # lc_index out of range (found on device)
    assert e.value.code == -4
    rr.rr_set_data(gm.ctx, t, lc, [0], [1], [0.0])
    gm.npt = 10
    gm.build_ld_table(np.ones((3, 1, 100)))
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_evaluate(gm.ctx, pv, flux)               # table npv 3 != 2
    assert e.value.code == -5
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_evaluate(gm.ctx, torch.zeros((3, 6), dtype=torch.float64, device="cuda"), flux)
    assert e.value.code == -3
    with pytest.raises(rr.RoadRunnerError):
        rr.rr_create(ng=1)
    gm.close()


# ---- host-buffer path -----------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", [0, 1])
def test_host_path_equals_device_path(rr, precision):
    wl = workloads.make_workload(4, npv=700, npt=60000)      # > 1 chunk of 256 MB flux in fp64
    gm = gpu_model(rr, wl, precision)
    ldp = wl.ldp(gm.mu)
    gm.build_ld_table(ldp)
    dev, st_dev = gm.evaluate(wl.pv, want_status=True)
    status = np.empty(wl.npv, np.int32)
    host = gm.evaluate_host(ldp, wl.pv, status=status)
    assert np.array_equal(host, dev.cpu().numpy())
    assert np.array_equal(status, st_dev.cpu().numpy())
    gm.close()


# ---- full size, the launch configuration bench.py times ----------------------------------------------------
@pytest.mark.parametrize("config,precision", [(4, 0), (4, 1), (4, 2), (3, 0), (3, 1), (2, 0), (2, 1),
                                              (1, 0)])
def test_full_size_sampled(rr, config, precision):
    """Full BASELINE size on the GPU; the oracle recomputes sampled (pv, exposure) pairs."""
    wl = workloads.make_workload(config)
    gm = gpu_model(rr, wl, precision)
    gm.build_ld_table(wl.ldp(gm.mu))
    flux = gm.evaluate(wl.pv)
    rng = np.random.default_rng(100 + config)
    pvs = np.sort(rng.choice(wl.npv, 48, replace=False))
    cols = np.sort(rng.choice(wl.npt, 1500, replace=False))
    # add exposures around each sampled pv's conjunction so that in-transit points are covered
    t0 = wl.pv[pvs, 1]
    near = np.unique(np.concatenate([np.argsort(np.abs(wl.times - t))[:40] for t in t0[:8]]))
    cols = np.unique(np.concatenate([cols, near]))
    import torch
    got = flux[torch.as_tensor(pvs, device="cuda")][:, torch.as_tensor(cols, device="cuda")] \
        .cpu().numpy().astype(np.float64)
    # property that holds at any size: flux <= 1, finite
    assert bool(torch.isfinite(flux).all()) and float(flux.max()) <= 1.0
    sub = wl.subset_pv(pvs).subset_times(cols)
    want, _ = oracle_flux(sub)
    tol = {0: TOL64, 1: TOL32, 2: 2e-8}[precision]
    assert np.max(np.abs(got - want)) <= tol
    assert (want < 1).sum() > 50
    gm.close()


# ---- round 2: the corners the first round left untested -----------------------------------------------
def _multiscale_times(span=2.0, n_log=900, n_lin=500):
    """Offsets from t0 = 0 on every scale from 1e-6 d to the span (both signs) plus a coarse uniform
    grid: resolves a 30 s periastron transit and a day-long apastron transit in one time axis."""
    lg = np.logspace(-6.0, np.log10(span), n_log)
    return np.sort(np.concatenate([-lg, [0.0], lg, np.linspace(-span, span, n_lin)]))


def _eccentric_population(e, rng, k_lo=0.03, k_hi=0.19):
    """One pv per argument of periastron over a full turn (w = pi/2: transit at periastron,
    w = 3pi/2: at apastron), impact parameters from central to grazing; t0 = 0."""
    ws = np.concatenate([np.linspace(0.0, 2 * np.pi, 16, endpoint=False), [0.5 * np.pi + 1e-3,
                                                                           1.5 * np.pi - 1e-3]])
    n = ws.size
    k = rng.uniform(k_lo, k_hi, n)
    a = (1.5 + k) / (1.0 - e) * rng.uniform(1.0, 1.5, n)
    b = rng.uniform(0.0, 1.0, n) * (1.0 + k)
    b[::5] = (1.0 + k[::5]) * 0.999                          # grazing
    b[1::5] = 0.0                                            # central
    p = rng.uniform(2.0, 4.0, n)
    cosi = b * (1.0 + e * np.sin(ws)) / (a * (1.0 - e * e))
    assert np.all(cosi < 1.0)
    return np.stack([k, np.zeros(n), p, a, np.arccos(cosi), np.full(n, e), ws], axis=1)


@pytest.mark.parametrize("e", [0.8, 0.9, 0.95, 0.99])
@pytest.mark.parametrize("precision,mode", [(0, 0), (0, 2), (1, 0), (1, 2), (2, 0)])
def test_flux_high_eccentricity(rr, e, precision, mode):
    """rr_evaluate (transit window + fast Halley path + robust solver) for e up to 0.99, w over a
    full turn, transits at periastron and at apastron, ns = 1 and 7, in the lazy and direct table
    modes (the ABI accepts any e < 1)."""
    rng = np.random.default_rng(int(e * 1000))
    pv = _eccentric_population(e, rng)
    t1 = _multiscale_times()
    times = np.concatenate([t1, t1])
    lc = np.repeat(np.arange(2, dtype=np.int32), t1.size)
    pbs, nss, ets = [0, 0], [1, 7], [0.0, 0.004]
    mc = workloads.ModelConfig()
    coeffs = np.tile(np.array([[[0.45, 0.15]]]), (pv.shape[0], 1, 1))
    if mode == 2:
        om = oracle.OracleDirectModel.from_config(mc)
        want, st_o = om.evaluate(times, lc, pbs, nss, ets, pv,
                                 workloads.sample_profile("quadratic", coeffs, om.mu), nthreads=0)
    else:
        om = oracle.OracleModel.from_config(mc)
        om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
        want, st_o = om.evaluate(times, lc, pbs, nss, ets, pv, nthreads=0)
    gm = rr.RoadRunner.from_config(mc, precision)
    rr.rr_set_table_mode(gm.ctx, mode)
    gm.set_data(times, lc, pbs, nss, ets)
    gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
    got, st = gm.evaluate(pv, want_status=True)
    got = got.cpu().numpy().astype(np.float64)
    assert np.array_equal(st.cpu().numpy(), st_o) and not st_o.any()
    # every pv is sampled inside its transit, in both light curves
    assert np.all((want[:, :t1.size] < 1).sum(axis=1) > 20)
    assert np.all((want[:, t1.size:] < 1).sum(axis=1) > 20)
    err = np.max(np.abs(got - want), axis=1)
    # RR_MIXED: z carries ~3 eps32 relative, d(deficit)/dz <= ~0.2 for k <= 0.3 -> 4e-8, plus the
    # fp32 rounding of ip*ap (<= 1e-8): 5e-8 derived; measured here <= 2.1e-8
    tol = {0: TOL64, 1: TOL32, 2: 5e-8}[precision]
    assert np.max(err) <= tol, (e, precision, mode, [float(f"{x:.2e}") for x in err])
    gm.close()


@pytest.mark.parametrize("precision", [0, 1])
def test_direct_model_large_radius_ratios(rr, precision):
    """RR_TABLE_DIRECT accepts any k > 0 (roadrunner.h): k^2 > 1/2, k just below / at / above 1
    (planet as large as or larger than the star: afull = pi min(1,k)^2, |1-k|), circular and
    eccentric, against the oracle's direct model."""
    ks = np.array([0.45, 0.72, 0.999, 1.0, 1.001, 1.5, 0.9, 1.2])
    n = ks.size
    rng = np.random.default_rng(77)
    e = np.where(np.arange(n) % 2 == 0, 0.0, rng.uniform(0.1, 0.6, n))
    w = rng.uniform(0, 2 * np.pi, n)
    a = (1.6 + ks) / (1 - e) * rng.uniform(1.0, 1.6, n)
    b = rng.uniform(0.0, 1.0, n) * (1 + ks)
    b[2:5] = [0.0, 0.3, 1.9]
    cosi = b * (1 + e * np.sin(w)) / (a * (1 - e * e))
    pv = np.stack([ks, np.zeros(n), rng.uniform(2, 5, n), a, np.arccos(cosi), e, w], axis=1)
    t1 = np.linspace(-0.6, 0.6, 3001)
    times = np.concatenate([t1, t1])
    lc = np.repeat(np.arange(2, dtype=np.int32), t1.size)
    pbs, nss, ets = [0, 0], [1, 5], [0.0, 0.01]
    mc = workloads.ModelConfig()
    coeffs = np.tile(np.array([[[0.5, 0.2]]]), (n, 1, 1))
    om = oracle.OracleDirectModel.from_config(mc)
    want, st_o = om.evaluate(times, lc, pbs, nss, ets, pv,
                             workloads.sample_profile("quadratic", coeffs, om.mu), nthreads=0)
    rows_o, _ = om.rows(workloads.sample_profile("quadratic", coeffs, om.mu), pv)
    gm = rr.RoadRunner.from_config(mc, precision)
    rr.rr_set_table_mode(gm.ctx, rr.RR_TABLE_DIRECT)
    gm.set_data(times, lc, pbs, nss, ets)
    gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
    got, st = gm.evaluate(pv, want_status=True)
    got = got.cpu().numpy().astype(np.float64)
    rows_g = gm.rows().astype(np.float64)
    assert np.array_equal(st.cpu().numpy(), st_o) and not st_o.any()
    assert np.max(np.abs(rows_g - rows_o)) <= (3e-7 if precision else 1e-12)
    assert np.all((want < 1).sum(axis=1) > 100)
    assert want.min() < 0.05                                  # a k >= 1 planet hides the star
    err = np.max(np.abs(got - want), axis=1)
    # fp32: the occulted light ip*ap is rounded in fp32, so its error scales with the transit depth
    # ~k^2; the north-star's 2e-7 is stated for k <= 0.3 and is scaled by (k/0.3)^2 above that,
    # capped at the k = 1 value (parity bars)
    tol = TOL32 * np.maximum(1.0, np.minimum(ks, 1.0) ** 2 / 0.09) if precision else TOL64
    assert np.all(err <= tol), [float(f"{x:.2e}") for x in err]
    gm.close()


def test_orbit_z_fp64_on_an_fp32_ctx(rr):
    """roadrunner.h: rr_orbit_z(fp32_math = 0) is fp64 in both precisions of ctx (the Halley
    acceptance tolerance follows the arithmetic asked for, not the ctx precision)."""
    wl = workloads.make_workload(4, npv=24, npt=1500)
    _, _, z_o = oracle.evaluate_workload(wl, want_z=True)
    for precision in (1, 2):
        gm = gpu_model(rr, wl, precision)
        z_g = gm.orbit_z(wl.pv).cpu().numpy()
        assert np.max(np.abs(z_g - z_o)) <= 1e-11 * max(1.0, float(np.max(np.abs(z_o))))
        gm.close()


def test_pv_shards_concatenate_to_the_whole(rr):
    """the path shards on the pv axis with no exchange.  The two shard.pv_slice halves
    of one population, evaluated separately on one device, equal the whole bit for bit."""
    from paper_2009_08500_b200 import shard
    wl = workloads.make_workload(3, npv=257, npt=6 * 500)
    for precision in (0, 1):
        gm = gpu_model(rr, wl, precision)
        # RR_REDUCE_AUTO picks the supersample layout from npv x npt (the amount of work), and the
        # two layouts sum the sub-samples in different orders: bitwise equality across shardings
        # needs the layout pinned
        rr.rr_set_reduction(gm.ctx, rr.RR_REDUCE_THREAD)
        ldp = wl.ldp(gm.mu)
        gm.build_ld_table(ldp)
        whole, st_w = gm.evaluate(wl.pv, want_status=True)
        whole, st_w = whole.cpu().numpy(), st_w.cpu().numpy()
        parts, sts = [], []
        for r in range(2):
            b, e_ = shard.pv_slice(wl.npv, r, 2)
            gm.build_ld_table(ldp[b:e_])
            f, st = gm.evaluate(wl.pv[b:e_], want_status=True)
            parts.append(f.cpu().numpy())
            sts.append(st.cpu().numpy())
        assert np.array_equal(np.concatenate(parts), whole)
        assert np.array_equal(np.concatenate(sts), st_w)
        rr.rr_set_reduction(gm.ctx, rr.RR_REDUCE_AUTO)           # ... and to rounding without
        b, e_ = shard.pv_slice(wl.npv, 1, 2)
        gm.build_ld_table(ldp[b:e_])
        auto = gm.evaluate(wl.pv[b:e_]).cpu().numpy()
        assert np.max(np.abs(auto.astype(np.float64) - whole[b:e_])) <= (2e-7 if precision else 1e-14)
        gm.close()


def test_binding_rejects_wrong_dtype_and_size(rr):
    """A tensor of the wrong dtype or size never reaches the kernels (it would be an out-of-bounds
    device read or write): TypeError / ValueError from the binding."""
    import torch
    wl = workloads.make_workload(1, npv=4, npt=300)
    gm = gpu_model(rr, wl, rr.RR_FP64)
    ldp64 = torch.as_tensor(wl.ldp(gm.mu)).cuda()
    with pytest.raises(TypeError):
        rr.rr_build_ld_table(gm.ctx, ldp64.float(), 4)           # fp32 profile, fp64 ctx
    with pytest.raises(ValueError):
        rr.rr_build_ld_table(gm.ctx, ldp64[:3].contiguous(), 4)  # 3 profiles for npv = 4
    rr.rr_build_ld_table(gm.ctx, ldp64, 4)
    pv = torch.as_tensor(wl.pv).cuda()
    with pytest.raises(ValueError):
        rr.rr_evaluate(gm.ctx, pv, torch.empty((4, 299), dtype=torch.float64, device="cuda"))
    with pytest.raises(TypeError):
        rr.rr_evaluate(gm.ctx, pv, torch.empty((4, 300), dtype=torch.float32, device="cuda"))
    flux = torch.empty((4, 300), dtype=torch.float64, device="cuda")
    with pytest.raises(ValueError):
        rr.rr_evaluate(gm.ctx, pv, flux, torch.empty(3, dtype=torch.int32, device="cuda"))
    with pytest.raises(TypeError):
        rr.rr_evaluate(gm.ctx, pv, flux, torch.empty(4, dtype=torch.int64, device="cuda"))
    rr.rr_evaluate(gm.ctx, pv, flux)
    ref = flux.cpu().numpy()
    gm.build_ld_table(ldp64.float())                             # the wrapper casts to the ctx dtype
    assert np.max(np.abs(gm.evaluate(wl.pv).cpu().numpy() - ref)) <= 1e-7
    gm.close()
    g32 = gpu_model(rr, wl, rr.RR_FP32)
    with pytest.raises(TypeError):
        rr.rr_build_ld_table(g32.ctx, ldp64, 4)                  # fp64 profile, fp32 ctx
    with pytest.raises(TypeError):
        rr.rr_evaluate_host(g32.ctx, wl.ldp(g32.mu), wl.pv, np.empty((4, 300), np.float32))
    g32.close()


def test_named_law_build_is_asynchronous_and_repeatable(rr):
    """rr_build_ld_table_law queues its work on the caller's stream (no allocation, no host
    round trip after the first call): many back-to-back builds + evaluations on a side stream give
    the same flux as one synchronous pass."""
    import torch
    mc = workloads.ModelConfig()
    base = workloads.make_workload(1, npv=64, npt=800)
    gm = gpu_model(rr, base)
    rng = np.random.default_rng(4)
    ldcs = [torch.as_tensor(np.stack([rng.uniform(0.1, 0.6, (64, 1)), rng.uniform(0.0, 0.3, (64, 1))],
                                     axis=-1)).cuda() for _ in range(6)]
    pv = torch.as_tensor(base.pv).cuda()
    ref = []
    for ldc in ldcs:
        rr.rr_build_ld_table_law(gm.ctx, "quadratic", ldc, 64)
        ref.append(gm.evaluate(pv).clone())
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    outs = [torch.empty_like(ref[0]) for _ in ldcs]
    with torch.cuda.stream(side):
        for ldc, out in zip(ldcs, outs):
            rr.rr_build_ld_table_law(gm.ctx, "quadratic", ldc, 64)
            rr.rr_evaluate(gm.ctx, pv, out)
    side.synchronize()
    for a, b in zip(ref, outs):
        assert torch.equal(a, b)
    gm.close()


# ---- the device math of the hot path, function by function (rr_math.cuh through rr_math_probe) ----------
def _mp_vec(f, *cols):
    import mpmath as mp
    mp.mp.dps = 40
    return np.array([float(f(*[mp.mpf(float(x)) for x in row])) for row in zip(*cols)])


@pytest.mark.parametrize("fp32", [False, True])
def test_device_math_against_multiprecision(rr, fp32):
    """rr_sqrt3 / rr_sqrt / rr_div3 / rr_rcp / rr_atan_t / rr_atan_quadrant / rr_atan2_pos /
    rr_sincosm1_small / rr_cell on the ranges the kernels use them on, against 40-digit arithmetic:
    fp64 within a few ulp, fp32 within a few fp32 ulp (the bounds DESIGN.md s6 states)."""
    import mpmath as mp
    import torch
    rng = np.random.default_rng(31)
    n = 4000
    ulp = 2.0 ** -23 if fp32 else 2.0 ** -52

    def dev(x):
        x = np.asarray(x, np.float64)
        if fp32:
            x = x.astype(np.float32).astype(np.float64)        # the probe rounds its inputs to fp32
        return x, torch.as_tensor(x).cuda()

    def run(op, a, b=None):
        o0, o1 = rr.rr_math_probe(op, a, b, fp32_math=fp32)
        return o0.cpu().numpy(), o1.cpu().numpy()

    # square roots: z^2 from 1e-12 to 1e4, and exact squares
    x, xd = dev(np.concatenate([10.0 ** rng.uniform(-12, 4, n), np.arange(1.0, 30.0) ** 2]))
    want = _mp_vec(mp.sqrt, x)
    for op in ("sqrt3", "sqrt"):
        got, _ = run(op, xd)
        assert np.max(np.abs(got / want - 1.0)) <= 2.0 * ulp, op
    got, _ = run("sqrt", torch.as_tensor(np.array([0.0, -1.0, -1e-300])).cuda())
    assert np.array_equal(got, np.zeros(3))
    # division and reciprocal
    a, ad = dev(rng.uniform(-3, 3, n))
    b, bd = dev(10.0 ** rng.uniform(-6, 3, n))
    got, _ = run("div3", ad, bd)
    assert np.max(np.abs(got - _mp_vec(lambda p, q: p / q, a, b)) / np.maximum(np.abs(a / b), 1e-300)) \
        <= 2.0 * ulp
    got, _ = run("rcp", bd)
    assert np.max(np.abs(got * b - 1.0)) <= (3e-7 if fp32 else 1e-11)
    # atan on the reduced range, a little beyond it, and near zero
    T = float(mp.tan(mp.pi / 8))
    t, td = dev(np.concatenate([rng.uniform(-T, T, n), [T * (1 + 2e-7), -T, 0.0, 1e-9, 1e-300]]))
    got, _ = run("atan_t", td)
    want = _mp_vec(mp.atan, t)
    assert np.max(np.abs(got - want)) <= 1.5 * ulp * 0.5          # |atan| < 0.4: 1.5 ulp of 0.25..0.5
    # the lens half-angles: atan(sqrt(P/S)) from (S, P), every octant, the octant boundaries, P = 0
    S, Sd = dev(np.concatenate([10.0 ** rng.uniform(-8, 1, n), [1.0, 1.0, 1.0, 2.0, 3.0]]))
    P, Pd = dev(np.concatenate([10.0 ** rng.uniform(-8, 1, n),
                                [0.0, T * T, 1.0 / (T * T), 2.0, 1e-30]]))
    got, _ = run("atan_quadrant", Sd, Pd)
    want = _mp_vec(lambda s_, p_: mp.atan(mp.sqrt(p_ / s_)), S, P)
    assert np.max(np.abs(got - want)) <= (6.0 if fp32 else 4.0) * ulp
    # atan2 for y >= 0 (direct-model rows)
    y, yd = dev(np.concatenate([10.0 ** rng.uniform(-8, 1, n), [0.0, 1.0, 1.0]]))
    xx, xxd = dev(np.concatenate([rng.uniform(-3, 3, n), [1.0, 0.0, -1.0]]))
    got, _ = run("atan2_pos", yd, xxd)
    want = _mp_vec(mp.atan2, y, xx)
    assert np.max(np.abs(got - want)) <= (8.0 if fp32 else 4.0) * ulp
    # sin, cos - 1 on |x| <= 0.5: relative accuracy (what the d = E - E_tr formulation relies on)
    d, dd = dev(np.concatenate([rng.uniform(-0.5, 0.5, n), 10.0 ** rng.uniform(-12, -1, 500),
                                [0.5, -0.5, 0.0]]))
    s_g, c_g = run("sincosm1", dd)
    s_w, c_w = _mp_vec(mp.sin, d), _mp_vec(lambda v: mp.cos(v) - 1, d)
    nz = d != 0
    assert np.max(np.abs(s_g[nz] / s_w[nz] - 1.0)) <= 2.0 * ulp
    assert np.max(np.abs(c_g[nz] / c_w[nz] - 1.0)) <= 2.5 * ulp
    assert s_g[~nz].item() == 0.0 and c_g[~nz].item() == 0.0
    # table cell: floor and fractional part, exact
    yv, yvd = dev(np.concatenate([rng.uniform(0, 5000, n), [0.0, 98.99999999999999, 99.0, 4999.5]]))
    ig, ag = run("cell", yvd)
    assert np.array_equal(ig, np.floor(yv)) and np.array_equal(ag, yv - np.floor(yv))


def test_dispatch_million_exposures(rr):
    """Kernel 4 on 1.2e6 exposures in 4000 runs of random lengths (the run heads are found by many
    blocks: their per-block counts, a scan, a scatter): bit-exact against the restatement."""
    rng = np.random.default_rng(17)
    nlc = 5
    cuts = np.sort(rng.choice(np.arange(1, 1_200_000), 3999, replace=False))
    lens = np.diff(np.concatenate([[0], cuts, [1_200_000]]))
    ids = rng.integers(0, nlc, lens.size)
    ids[1:][ids[1:] == ids[:-1]] = (ids[:-1][ids[1:] == ids[:-1]] + 1) % nlc   # neighbours differ
    lc = np.repeat(ids, lens).astype(np.int32)
    times = rng.uniform(-10, 10, lc.size)
    ns = [1, 3, 7, 30, 2]
    gm = rr.RoadRunner(npb=2)
    gm.set_data(times, lc, [0, 1, 0, 1, 0], ns, [0.0, 0.01, 0.02, 0.03, 0.001])
    got = rr.rr_get_tiles(gm.ctx)
    want = expected_tiles(lc, ns, times)
    assert rr.rr_num_tiles(gm.ctx) == len(want)
    assert np.array_equal(got["start"], [w[0] for w in want])
    assert np.array_equal(got["count"], [w[1] for w in want])
    assert np.array_equal(got["lc"], [w[2] for w in want])
    for j in rng.choice(len(want), 200, replace=False):
        s0, c, _ = want[j]
        assert got["tmin"][j] == times[s0:s0 + c].min() and got["tmax"][j] == times[s0:s0 + c].max()
    assert rr.rr_num_subsamples(gm.ctx) == int(np.asarray(ns)[lc].sum())
    bad = lc.copy()
    bad[777_777] = nlc
    import torch
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_set_data(gm.ctx, torch.as_tensor(times).cuda(), torch.as_tensor(bad).cuda(),
                       [0, 1, 0, 1, 0], ns, [0.0] * 5)
    assert e.value.code == -4
    gm.close()


def test_step_is_cuda_graph_capturable(rr):
    """rr_build_ld_table + rr_evaluate make no allocation, host round trip or synchronisation in steady
    state (buffers grow only when a larger npv arrives), so a step can be captured into a CUDA graph
    and replayed: same flux, also after the inputs changed in place."""
    import torch
    wl = small_workload(3)
    gm = gpu_model(rr, wl)
    ldp = torch.as_tensor(wl.ldp(gm.mu)).cuda()
    pv = torch.as_tensor(wl.pv).cuda()
    flux = torch.empty((wl.npv, wl.npt), dtype=torch.float64, device="cuda")
    status = torch.empty(wl.npv, dtype=torch.int32, device="cuda")

    def step():
        rr.rr_build_ld_table(gm.ctx, ldp, wl.npv)
        rr.rr_evaluate(gm.ctx, pv, flux, status)

    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        step()                                   # warm-up: every buffer has its size
        torch.cuda.synchronize()
        with torch.cuda.graph(graph, stream=side):
            step()
    want, _ = oracle_flux(wl)
    flux.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert np.max(np.abs(flux.cpu().numpy() - want)) <= TOL64
    pv2 = wl.pv.copy()
    pv2[:, 0] = np.clip(pv2[:, 0] * 1.07, 0.02, 0.2)          # new radius ratios, same buffers
    pv.copy_(torch.as_tensor(pv2))
    graph.replay()
    torch.cuda.synchronize()
    wl.pv = pv2
    want2, _ = oracle_flux(wl)
    assert np.max(np.abs(flux.cpu().numpy() - want2)) <= TOL64
    assert np.max(np.abs(want2 - want)) > 1e-5
    gm.close()


def test_lens_polynomial_radius_ratio_edges(rr):
    """The fp64 kernel takes the lens area between the contacts from per-pv polynomials for k <= 0.32
    and from the two-arctangent form above: radius ratios from 0.005 to just past the switch, in the
    direct model (any k > 0), ingress and egress densely sampled (2e-5 d steps), central to grazing
    impact parameters; flux against the oracle, which only knows the arctangent form.  The observed
    agreement is ~1e-14 on both sides of the switch."""
    ks = np.array([0.005, 0.01, 0.05, 0.15, 0.3, 0.3199, 0.32, 0.3201, 0.35, 0.5])
    n = ks.size
    rng = np.random.default_rng(5)
    e = np.where(np.arange(n) % 2 == 0, 0.0, rng.uniform(0.1, 0.5, n))
    w = rng.uniform(0, 2 * np.pi, n)
    a = rng.uniform(6.0, 12.0, n)
    b = np.array([0.0, 0.5, 0.9, 0.3, 0.7, 0.1, 0.6, 0.95, 0.2, 1.2])
    cosi = b * (1 + e * np.sin(w)) / (a * (1 - e * e))
    pv = np.stack([ks, np.zeros(n), rng.uniform(2.5, 4.0, n), a, np.arccos(cosi), e, w], axis=1)
    t1 = np.arange(-0.16, 0.16, 2e-5)
    times = np.concatenate([t1, t1[::7]])
    lc = np.concatenate([np.zeros(t1.size), np.ones(t1[::7].size)]).astype(np.int32)
    pbs, nss, ets = [0, 0], [1, 3], [0.0, 0.002]
    mc = workloads.ModelConfig()
    coeffs = np.tile(np.array([[[0.35, 0.25]]]), (n, 1, 1))
    om = oracle.OracleDirectModel.from_config(mc)
    want, _ = om.evaluate(times, lc, pbs, nss, ets, pv,
                          workloads.sample_profile("quadratic", coeffs, om.mu), nthreads=0)
    gm = rr.RoadRunner.from_config(mc)
    rr.rr_set_table_mode(gm.ctx, rr.RR_TABLE_DIRECT)
    gm.set_data(times, lc, pbs, nss, ets)
    gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
    got = gm.evaluate(pv).cpu().numpy()
    err = np.max(np.abs(got - want), axis=1)
    assert np.all((want < 1).sum(axis=1) > 1000)
    assert np.max(err) <= TOL64, [float(f"{x:.1e}") for x in err]
    assert np.max(err) <= 1e-12, [float(f"{x:.1e}") for x in err]      # what the arithmetic gives
    gm.close()


def test_orbit_polynomials_against_the_per_subsample_solve(rr):
    """rr_set_orbit_poly: the fp64 kernel takes z^2 of eccentric pvs from per-pv polynomials over the
    transit window (fitted through 26 exact Kepler solves per evaluate) where they converge, and solves
    Kepler's equation per sub-sample otherwise.  Both against the oracle (which always solves), the two
    against each other, and the class counters: most of config 3's / 4's eccentric sub-samples go
    through the polynomials, none with the switch off, none for e = 0.99 at periastron (no
    convergence: the gate must send those to the solver)."""
    for config in (3, 4):
        wl = small_workload(config)
        want, _ = oracle_flux(wl)
        gm = gpu_model(rr, wl)
        gm.build_ld_table(wl.ldp(gm.mu))
        out = {}
        for on in (True, False):
            rr.rr_set_orbit_poly(gm.ctx, on)
            rr.rr_enable_counters(gm.ctx, True)
            out[on] = gm.evaluate(wl.pv).cpu().numpy()
            cnt = rr.rr_get_counters(gm.ctx)
            rr.rr_enable_counters(gm.ctx, False)
            assert np.max(np.abs(out[on] - want)) <= 1e-12
            if on:
                assert cnt["eccentric_poly"] > 0.5 * cnt["eccentric"] > 0
            else:
                assert cnt["eccentric_poly"] == 0 and cnt["solver_iters"] >= cnt["eccentric"] > 0
        assert 0 < np.max(np.abs(out[True] - out[False])) <= 1e-12
        gm.close()
    # gate: wide windows of close-in, very eccentric orbits do not converge
    rng = np.random.default_rng(990)
    pv = _eccentric_population(0.99, rng)
    t1 = _multiscale_times()
    mc = workloads.ModelConfig()
    coeffs = np.tile(np.array([[[0.45, 0.15]]]), (pv.shape[0], 1, 1))
    gm = rr.RoadRunner.from_config(mc)
    gm.set_data(t1, np.zeros(t1.size, np.int32), [0], [1], [0.0])
    gm.build_ld_table(workloads.sample_profile("quadratic", coeffs, gm.mu))
    rr.rr_enable_counters(gm.ctx, True)
    gm.evaluate(pv)
    cnt = rr.rr_get_counters(gm.ctx)
    assert 0 < cnt["eccentric"] and cnt["eccentric_poly"] < cnt["eccentric"]
    gm.close()


@pytest.mark.parametrize("precision", [0, 1])
def test_lens_polynomials_against_the_exact_lens_area(rr, precision):
    """rr_set_lens_poly: the area between the contacts from per-(pv, k) polynomials (default) or from
    the two-arctangent form per sub-sample; both against the oracle and against each other."""
    wl = small_workload(4)
    want, _ = oracle_flux(wl)
    gm = gpu_model(rr, wl, precision)
    gm.build_ld_table(wl.ldp(gm.mu))
    out = {}
    for on in (True, False):
        rr.rr_set_lens_poly(gm.ctx, on)
        out[on] = gm.evaluate(wl.pv).cpu().numpy().astype(np.float64)
        assert np.max(np.abs(out[on] - want)) <= (TOL32 if precision else 1e-12)
    d = np.max(np.abs(out[True] - out[False]))
    assert 0 < d <= (2e-7 if precision else 1e-12)
    gm.close()


def test_bench_line_contract(rr):
    """bench.py prints ONE JSON line with the keys the driver reads (a small population here; the
    default run uses config 4 at full size)."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--config", "3", "--npv", "96",
                          "--npt", "6000", "--steps", "3", "--warmup", "3", "--no-all-configs"],
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.strip().splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
                "higher_is_better", "scaling", "vs_baseline", "dtype", "data", "config", "clocks",
                "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in d, key
    assert d["unit"] == "evaluations/s" and d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3
    assert d["higher_is_better"] is True and d["vs_baseline"] is None and d["dtype"] == "f64"
    assert d["config"]["workload"] == "config3-heterogeneous" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["gpu_launches"] >= 3 * 5
    assert abs(d["value"] - d["config"]["evaluations_per_step_per_gpu"] / (d["ms_per_step"] * 1e-3)) \
        <= 1e-6 * d["value"]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] >= 96 * 6000 * 8
    r = d["roofline"]
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel_ms", "counter_based",
                "executed_frac_by_table", "class_counts"):
        assert key in r, key
    assert r["bound"] in ("hbm", "alu") and 0 < r["frac"] and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["value"] > 0 and c["cores"] >= 1 and c["sample"]
    assert c["one_thread"] > 0 and c["all_cores"] > 0 and c["cpu_model"]
    assert d["max_abs_err_vs_oracle_sample"]["value"] <= TOL64
