"""Pins for the oracle's DIRECT model: weights at the pv's own
k, g interpolation only.  CPU only."""
import math

import numpy as np

import oracle
import workloads
from oracle import truth


def test_direct_row_on_g_nodes_equals_l1():
    """At z = g_ig (1+k) the interpolation weight is 0: flux from the row is Eq. (5) with the weight
    vector at exactly that (c, k) - the L1 function, which is pinned against Eq. (2)."""
    m = oracle.OracleDirectModel()
    ld = truth.quadratic(0.4, 0.2)(m.mu)
    for k in (0.013, 0.1, 0.27, 0.5):
        pv = np.array([[k, 0, 3, 8, 1.5, 0, 0]])
        rows, ist = m.rows(ld, pv)
        for ig in range(0, m.ng - 1, 7):
            c = ig / (m.ng - 1) * (1 + k)
            assert abs(oracle.flux_from_row(c, k, rows[0, 0], ist[0, 0])
                       - oracle.direct_flux(k, c, m.ze, ld, ist[0, 0])) < 1e-15


def test_direct_uniform_disc_exact():
    """ldp = 1: every weight vector sums to 1, the row is 1, flux = 1 - a(z,k)/pi."""
    m = oracle.OracleDirectModel()
    ld = np.ones(m.nz)
    for k in (0.05, 0.3):
        rows, ist = m.rows(ld, np.array([[k, 0, 3, 8, 1.5, 0, 0]]))
        assert np.max(np.abs(rows - 1.0)) < 1e-13
        assert ist[0, 0] == np.pi or abs(ist[0, 0] - math.pi) < 1e-15
        for z in np.linspace(0, 1 + k, 23):
            want = 1 - oracle.lens_area(1.0, k, z) / math.pi
            assert abs(oracle.flux_from_row(z, k, rows[0, 0], ist[0, 0]) - want) < 1e-14


def test_direct_last_node_is_limb_sample_and_rows_are_dot_products():
    m = oracle.OracleDirectModel(nzin=7, nzlimb=5, ng=11)
    rng = np.random.default_rng(2)
    ld = rng.uniform(0.2, 1.0, m.nz)
    k = 0.17
    rows, _ = m.rows(ld, np.array([[k, 0, 3, 8, 1.5, 0, 0]]))
    assert rows[0, 0, -1] == ld[-1]                               # reading R5
    for ig in range(m.ng - 1):
        w = oracle.weights(ig / (m.ng - 1) * (1 + k), k, m.ze)
        assert abs(rows[0, 0, ig] - float(np.dot(w, ld))) < 1e-15


def test_direct_is_closer_to_l0_than_the_interpolated_model():
    """No k interpolation: 'small reduction in accuracy' of the interpolated model
    read the other way round.  Both against Eq. (2) by 20-digit quadrature."""
    ldf = truth.quadratic(0.4, 0.2)
    md, mi = oracle.OracleDirectModel(), oracle.OracleModel()
    lib = oracle.load()
    k = 0.1037                                                     # between two k nodes
    rows, ist = md.rows(ldf(md.mu), np.array([[k, 0, 3, 8, 1.5, 0, 0]]))
    T, ist2 = mi.build_ld_table(ldf(mi.mu)[None, None, :])
    ed, ei = [], []
    for z in np.linspace(0, 1 + k, 31):
        want = float(truth.flux_radial_mp(k, z, ldf, dps=20))
        ed.append(abs(oracle.flux_from_row(z, k, rows[0, 0], ist[0, 0]) - want))
        ei.append(abs(lib.oracle_flux_from_table(z, k, T.ctypes.data_as(oracle._D), mi.nk, mi.k0,
                                                 mi.k1, mi.ng, ist2[0, 0]) - want))
    assert max(ed) < 12e-6 and np.mean(ed) < 1.5e-6
    assert np.mean(ed) <= np.mean(ei) * 1.05


def test_direct_evaluate_equals_table_model_on_a_k_node_and_allows_any_k():
    """On a k node of the table the interpolated model has ak = 0: both models use the same weight
    vectors, so whole light curves agree to rounding; k outside the table's range is fine."""
    wl = workloads.make_workload(3, npv=4, npt=6 * 50)
    mi = oracle.OracleModel.from_config(wl.model)
    dk = (mi.k1 - mi.k0) / (mi.nk - 1)
    wl.pv[:, 0] = mi.k0 + dk * np.array([3, 17, 30, 48])
    mi.build_ld_table(wl.ldp(mi.mu))
    want, _ = mi.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                          wl.exposure_time, wl.pv)
    md = oracle.OracleDirectModel.from_config(wl.model)
    got, st = md.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                          wl.exposure_time, wl.pv, wl.ldp(md.mu))
    assert np.all(st == 0) and np.max(np.abs(got - want)) < 1e-13 and (want < 1).sum() > 50
    pv = wl.pv.copy()
    pv[0, 0] = 0.45                    # above the table's k1 = 0.2
    pv[1, 0] = -0.1                    # invalid
    got, st = md.evaluate(wl.times, wl.lc_index, wl.passband_index, wl.supersampling,
                          wl.exposure_time, pv, wl.ldp(md.mu))
    assert list(st) == [0, 1, 0, 0] and np.all(np.isnan(got[1])) and np.all(np.isfinite(got[0]))
    assert got[0].min() < 0.9          # a k = 0.45 transit is deep


# ---- transmission-spectroscopy shortcut (reading R13) ------------------------------
def _chromatic_case(spread):
    mc = workloads.ModelConfig(npb=3, nkpb=3)
    rng = np.random.default_rng(8)
    base = workloads.make_workload(1, npv=5, npt=10).pv
    kk = np.clip(base[:, :1] * (1 + spread * rng.uniform(-1, 1, (5, 3))), 0.021, 0.199)
    pv = np.concatenate([kk, base[:, 1:]], axis=1)
    times = np.tile(np.linspace(-0.15, 0.15, 400), 3)
    lc = np.repeat(np.arange(3, dtype=np.int32), 400)
    coeffs = rng.uniform(0.1, 0.4, (5, 3, 2))
    return mc, pv, times, lc, coeffs


def test_mean_k_weights_equal_k_is_identity_and_small_otherwise():
    """All passbands at the same k: the shortcut changes nothing (exact).  With +-3 % of chromatic
    variation (large for transmission spectroscopy) it moves the flux by < 1e-4, most in
    ingress/egress and for grazing transits, where a planet of radius kbar and one of radius k sample
    different parts of the steep limb: the 'insignificant effect' of PAPER.md:190.  Not zero."""
    for spread, lo, hi in ((0.0, -1.0, 0.0), (0.03, 1e-12, 1e-4)):
        mc, pv, times, lc, coeffs = _chromatic_case(spread)
        for model in ("table", "direct"):
            if model == "table":
                om = oracle.OracleModel.from_config(mc)
                om.build_ld_table(workloads.sample_profile("quadratic", coeffs, om.mu))
                a, _ = om.evaluate(times, lc, [0, 1, 2], [1, 1, 2], [0.0, 0.0, 0.01], pv)
                b, _ = om.evaluate(times, lc, [0, 1, 2], [1, 1, 2], [0.0, 0.0, 0.01], pv,
                                   mean_k_weights=True)
            else:
                om = oracle.OracleDirectModel.from_config(mc)
                ldp = workloads.sample_profile("quadratic", coeffs, om.mu)
                a, _ = om.evaluate(times, lc, [0, 1, 2], [1, 1, 2], [0.0, 0.0, 0.01], pv, ldp)
                b, _ = om.evaluate(times, lc, [0, 1, 2], [1, 1, 2], [0.0, 0.0, 0.01], pv, ldp,
                                   mean_k_weights=True)
            d = float(np.max(np.abs(a - b)))
            assert lo < d <= hi, (spread, model, d)
            assert (a < 1).sum() > 100


# ---- small-planet approximation (reading R14) ---------------------------------------
def test_profile_at_is_the_library_interpolant():
    """oracle_profile_at = numpy.interp over the bin means (linear, constant beyond the end nodes)."""
    m = oracle.OracleDirectModel()
    rng = np.random.default_rng(4)
    ld = np.sort(rng.uniform(0.1, 1.0, m.nz))[::-1].copy()
    for z in np.concatenate([rng.uniform(0, 1.3, 300), m.zm[[0, 1, 50, -2, -1]], [0.0, 1.0]]):
        assert abs(oracle.profile_at(z, m.zm, ld) - float(np.interp(z, m.zm, ld))) < 1e-15


def test_small_planet_rows_and_threshold():
    """Rows with k <= threshold hold the profile at the planet's centre z = g (1+k); rows above the
    threshold are the direct-model rows, bit for bit."""
    m = oracle.OracleDirectModel()
    ld = truth.power2(0.6, 0.7)(m.mu)
    pv = np.array([[0.01, 0, 3, 8, 1.5, 0, 0], [0.05, 0, 3, 8, 1.5, 0, 0]])
    ldp = np.stack([ld, ld])[:, None, :]
    plain, _ = m.rows(ldp, pv)
    sp, _ = m.rows(ldp, pv, small_planet_k=0.02)
    assert np.array_equal(sp[1], plain[1])
    g = np.arange(m.ng) / (m.ng - 1)
    g[-1] = 1.0
    assert np.max(np.abs(sp[0, 0] - np.interp(g * 1.01, m.zm, ld))) < 1e-15
    assert sp[0, 0, -1] == ld[-1]                                  # centre beyond the limb: R5


def test_small_planet_is_close_to_the_direct_model_inside_the_disc():
    """'If the planet is small enough': k = 0.01, centre at z <= 0.8: the flux moves by < 5e-8
    (depth 1e-4); at the limb the approximation is poor, which is why it has a threshold."""
    m = oracle.OracleDirectModel()
    ld = truth.quadratic(0.4, 0.2)(m.mu)
    k = 0.01
    pv = np.array([[k, 0, 3, 8, 1.5, 0, 0]])
    a, ist = m.rows(ld, pv)
    b, _ = m.rows(ld, pv, small_planet_k=0.02)
    inner = max(abs(oracle.flux_from_row(z, k, a[0, 0], ist[0, 0])
                    - oracle.flux_from_row(z, k, b[0, 0], ist[0, 0])) for z in np.linspace(0, 0.8, 81))
    limb = max(abs(oracle.flux_from_row(z, k, a[0, 0], ist[0, 0])
                   - oracle.flux_from_row(z, k, b[0, 0], ist[0, 0])) for z in np.linspace(0.97, 1.009, 40))
    assert 0 < inner < 5e-8 and limb > inner


# ---- named laws: closed-form disc integrals against quadrature -----------------
LAW_CASES = [("uniform", []), ("linear", [0.6]), ("quadratic", [0.4, 0.2]),
             ("quadratic-tri", [0.36, 0.3]), ("general", [0.3, 0.2, -0.1]),
             ("nonlinear", [0.5, -0.2, 0.4, -0.1]), ("logarithmic", [0.6, 0.2]),
             ("power-2", [0.6, 0.7]), ("power-2-pm", [0.7, 0.45])]


def test_named_law_disc_integrals():
    """Istar = 2 pi int_0^1 mu I dmu in closed form ('integrated analytically') vs
    30-digit quadrature of the same callable; every law is 1 at the disc centre."""
    for name, c in LAW_CASES:
        f, ist = truth.law(name, c)
        assert abs(float(f(1.0)) - 1.0) < 1e-15
        assert abs(float(truth.istar_mp(f)) - ist) < 1e-14, name
    f, ist = truth.law("exponential", [0.5, 0.01])
    assert ist is None and float(f(0.5)) < 1.0


def test_rows_from_parameter_vectors_pick_the_right_radius_ratio():
    """oracle_direct_rows_pv (row selection of readings R12 / R13, in C since round 2): row (pv, pb)
    is built at the pv's k of that passband, or at the mean of the pv's radius ratios with
    mean_k_weights; a pv with a non-finite or non-positive k gets NaN rows.  Against rows built one
    at a time with the k chosen here (weights pinned elsewhere: to L1 on the g nodes)."""
    mc = workloads.ModelConfig(npb=3, nkpb=3, nzin=20, nzlimb=20, ng=17)
    om = oracle.OracleDirectModel.from_config(mc)
    rng = np.random.default_rng(2)
    npv = 5
    pv = np.zeros((npv, 9))
    pv[:, :3] = rng.uniform(0.05, 0.2, (npv, 3))
    pv[:, 3:] = [0.0, 3.0, 8.0, 1.5, 0.1, 0.3]
    pv[3, 1] = -0.1                                   # invalid rows
    pv[4, 2] = np.nan
    ldp = workloads.sample_profile("quadratic", rng.uniform(0.1, 0.4, (npv, 3, 2)), om.mu)
    one = oracle.OracleDirectModel(mc.nzin, mc.nzlimb, mc.zcut, mc.ng, npb=1, nkpb=1)
    for mean in (False, True):
        rows, _ = om.rows(ldp, pv, mean_k_weights=mean)
        assert rows.shape == (npv, 3, mc.ng)
        assert np.isnan(rows[3:]).all() and not np.isnan(rows[:3]).any()
        for v in range(3):
            for b in range(3):
                k = pv[v, :3].mean() if mean else pv[v, b]
                pv1 = np.array([[k, 0.0, 3.0, 8.0, 1.5, 0.1, 0.3]])
                want, _ = one.rows(ldp[v, b][None, None, :], pv1)
                assert np.array_equal(rows[v, b], want[0, 0])
    a, _ = om.rows(ldp, pv, mean_k_weights=False)
    b_, _ = om.rows(ldp, pv, mean_k_weights=True)
    assert np.max(np.abs(a[:3] - b_[:3])) > 1e-6      # the two selections differ
