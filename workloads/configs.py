"""The five synthetic workloads of BASELINE.json ``configs`` (recipe: DESIGN.md section 4).

Every draw comes from ``numpy.random.default_rng(2009085000 + config)`` (PCG64).  Candidates are
drawn in blocks of fixed column order ``k, a, b, p, t0, e, w, circular?`` and a candidate is
dropped as a whole when it breaks a rejection rule; the first ``npv`` survivors are kept.  LD
coefficients are drawn afterwards, per (pv, passband), each with its own rejection loop.

Parameter-vector row (the ABI's ``pv``): ``[k_0 .. k_{nkpb-1}, t0, p, a, i, e, w]`` - the argument
order of the paper's ``evaluate(k, ldc, t0, p, a, i, e, w)`` with ``ldc`` replaced
by the sampled profile ``ldp``.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np

SEED_BASE = 2009085000
CONFIG_NAMES = {
    0: "config0-single-lc",
    1: "config1-population",
    2: "config2-long-cadence",
    3: "config3-heterogeneous",
    4: "config4-stress",
}
VARIANT_NAMES = {"4b": "config4b-literal-cadence"}


@dataclass(frozen=True)
class ModelConfig:
    """Resolution of the model: what ``rr_create`` receives."""
    nzin: int = 50
    nzlimb: int = 50
    zcut: float = 0.7
    ng: int = 100
    nk: int = 50
    k0: float = 0.02
    k1: float = 0.2
    npb: int = 1
    nkpb: int = 1          # 1 = achromatic radius ratio, npb = chromatic

    @property
    def nz(self) -> int:
        return self.nzin + self.nzlimb


@dataclass
class Workload:
    name: str
    model: ModelConfig
    times: np.ndarray            # [npt] f64, mid-exposure times (days)
    lc_index: np.ndarray         # [npt] i32  (paper: lcids)
    passband_index: np.ndarray   # [nlc] i32  (paper: pbids)
    supersampling: np.ndarray    # [nlc] i32  (paper: nsamples)
    exposure_time: np.ndarray    # [nlc] f64  (paper: exptimes, days)
    pv: np.ndarray               # [npv][nkpb+6] f64
    ld_kind: str                 # 'uniform' | 'quadratic' | 'power2' | 'poly4'
    ld_coeffs: np.ndarray        # [npv][npb][ncoef] f64
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def npv(self) -> int:
        return int(self.pv.shape[0])

    @property
    def npt(self) -> int:
        return int(self.times.shape[0])

    @property
    def nlc(self) -> int:
        return int(self.passband_index.shape[0])

    @property
    def evaluations_per_pv(self) -> int:
        """sum over exposures of their supersampling factor."""
        return int(self.supersampling.astype(np.int64)[self.lc_index].sum())

    @property
    def evaluations(self) -> int:
        return self.npv * self.evaluations_per_pv

    def ldp(self, mu: np.ndarray) -> np.ndarray:
        """Sample the LD law at the model's mu grid -> [npv][npb][nz] f64."""
        return sample_profile(self.ld_kind, self.ld_coeffs, mu)

    def subset_pv(self, index) -> "Workload":
        index = np.asarray(index)
        return replace(self, pv=np.ascontiguousarray(self.pv[index]),
                       ld_coeffs=np.ascontiguousarray(self.ld_coeffs[index]))

    def subset_times(self, index) -> "Workload":
        index = np.asarray(index)
        return replace(self, times=np.ascontiguousarray(self.times[index]),
                       lc_index=np.ascontiguousarray(self.lc_index[index]))


def sample_profile(kind: str, coeffs: np.ndarray, mu: np.ndarray) -> np.ndarray:
    """The caller-side LD law l(mu), evaluated at ``mu[nz]``.

    coeffs [..., ncoef] -> [..., nz].  Laws: uniform 1; quadratic 1-u1(1-mu)-u2(1-mu)^2;
    power-2 1-c(1-mu^alpha); poly4 1+sum_{n=1..4} c_n (1-mu)^n (config 3's tabulated profile).
    """
    mu = np.asarray(mu, dtype=np.float64)
    c = np.asarray(coeffs, dtype=np.float64)[..., None, :]      # [..., 1, ncoef]
    m = mu[:, None]                                              # [nz, 1]
    if kind == "uniform":
        return np.ones(c.shape[:-2] + (mu.size,))
    if kind == "quadratic":
        return 1.0 - c[..., 0] * (1.0 - m[:, 0]) - c[..., 1] * (1.0 - m[:, 0]) ** 2
    if kind == "power2":
        return 1.0 - c[..., 0] * (1.0 - m[:, 0] ** c[..., 1])
    if kind == "poly4":
        x = 1.0 - m[:, 0]
        return 1.0 + c[..., 0] * x + c[..., 1] * x**2 + c[..., 2] * x**3 + c[..., 3] * x**4
    raise ValueError(f"unknown LD law {kind!r}")


# ------------------------------------------------------------------------------------------
# draws
# ------------------------------------------------------------------------------------------
def _draw_orbits(rng, npv, k_range, ecc_max, circular_fraction):
    """Rows [k, t0, p, a, i, e, w]; rejection: cos i > 1 or a(1-e) <= 1+k."""
    rows = []
    have = 0
    while have < npv:
        u = rng.random((max(npv, 256), 8))
        k = k_range[0] + (k_range[1] - k_range[0]) * u[:, 0]
        a = 4.0 + 16.0 * u[:, 1]
        b = (1.0 + k) * u[:, 2]
        p = 1.0 + 9.0 * u[:, 3]
        t0 = -0.01 + 0.02 * u[:, 4]
        e = ecc_max * u[:, 5]
        w = 2.0 * np.pi * u[:, 6]
        circ = u[:, 7] < circular_fraction
        e = np.where(circ, 0.0, e)
        w = np.where(circ, 0.0, w)
        cosi = b * (1.0 + e * np.sin(w)) / (a * (1.0 - e * e))
        ok = (cosi <= 1.0) & (a * (1.0 - e) > 1.0 + k)
        inc = np.arccos(np.clip(cosi, -1.0, 1.0))
        block = np.stack([k, t0, p, a, inc, e, w], axis=1)[ok]
        rows.append(block)
        have += block.shape[0]
    return np.ascontiguousarray(np.concatenate(rows)[:npv])


def _draw_quadratic(rng, n):
    out = np.empty((n, 2))
    todo = np.arange(n)
    while todo.size:
        u1 = 0.8 * rng.random(todo.size)
        u2 = -0.2 + 0.6 * rng.random(todo.size)
        ok = ~((1.0 - u1 - u2 < 0.0) | (u1 + 2.0 * u2 < 0.0))
        out[todo[ok], 0] = u1[ok]
        out[todo[ok], 1] = u2[ok]
        todo = todo[~ok]
    return out


def _single_lc(npt, ns, exptime):
    return (np.zeros(npt, np.int32), np.zeros(1, np.int32), np.array([ns], np.int32),
            np.array([exptime], np.float64))


def make_workload(config, npv: int | None = None, npt: int | None = None) -> Workload:
    """Build config 0..4.  ``npv``/``npt`` shrink the population / time axis for parity tests
    (same seed, same draw order: a smaller npv is a prefix of the full population).

    ``"4b"``: the labelled secondary workload of SURVEY 8(d): config 4's population with the
    literal reading of "2-minute cadence spacing" - 10^5 exposures spaced 2 min apart (138.9 d
    centred on t = 0) instead of 10^5 exposures over +-0.5 d.  More than 90 % of it is out of
    transit: it isolates the window test and the flux = 1 fill path."""
    if str(config) == "4b":
        wl = make_workload(4, npv=npv, npt=npt)
        n = wl.npt
        times = (np.arange(n, dtype=np.float64) - 0.5 * (n - 1)) * (2.0 / 1440.0)
        return replace(wl, name=VARIANT_NAMES["4b"], times=times,
                       note="literal 2-minute spacing of the exposures")
    config = int(config)
    rng = np.random.default_rng(SEED_BASE + config)
    name = CONFIG_NAMES[config]
    if config == 0:
        model = ModelConfig()
        n = npt or 1000
        times = np.linspace(-0.2, 0.2, n)
        pv = np.array([[0.1, 0.0, 3.0, 8.0, np.deg2rad(88.0), 0.0, 0.0]])
        ld = np.array([[[0.4, 0.2]]])
        lc, pb, ns, et = _single_lc(n, 1, 0.0)
        return Workload(name, model, times, lc, pb, ns, et, pv, "quadratic", ld)
    if config == 1:
        model = ModelConfig()
        n, m = npt or 5000, npv or 1024
        times = np.linspace(-0.25, 0.25, n)
        pv = _draw_orbits(rng, m, (0.02, 0.2), 0.0, 1.0)
        ld = _draw_quadratic(rng, m).reshape(m, 1, 2)
        lc, pb, ns, et = _single_lc(n, 1, 0.0)
        return Workload(name, model, times, lc, pb, ns, et, pv, "quadratic", ld)
    if config == 2:
        model = ModelConfig()
        n, m = npt or 20000, npv or 4096
        times = np.linspace(-0.25, 0.25, n)
        pv = _draw_orbits(rng, m, (0.02, 0.2), 0.0, 1.0)
        c = 0.3 + 0.6 * rng.random(m)
        alpha = 0.3 + 0.9 * rng.random(m)
        ld = np.stack([c, alpha], axis=1).reshape(m, 1, 2)
        lc, pb, ns, et = _single_lc(n, 10, 0.0204)
        return Workload(name, model, times, lc, pb, ns, et, pv, "power2", ld)
    if config == 3:
        model = ModelConfig(nzin=100, nzlimb=100, npb=4)
        per_lc, m = (npt or 48000) // 6, npv or 8192
        times = np.tile(np.linspace(-0.25, 0.25, per_lc), 6)
        lc = np.repeat(np.arange(6, dtype=np.int32), per_lc)
        pb = np.array([0, 1, 2, 3, 0, 1], np.int32)
        ns = np.array([1, 1, 5, 5, 10, 30], np.int32)
        et = np.array([0.000694, 0.000694, 0.006944, 0.006944, 0.0204, 0.020833])
        pv = _draw_orbits(rng, m, (0.02, 0.2), 0.5, 0.0)
        u = rng.random((m, 4, 4))
        ld = np.stack([-(0.2 + 0.4 * u[..., 0]), -(0.2 * u[..., 1]), -(0.1 * u[..., 2]),
                       -(0.05 * u[..., 3])], axis=-1)
        return Workload(name, model, times, lc, pb, ns, et, pv, "poly4", ld)
    if config == 4:
        model = ModelConfig(k0=0.01, k1=0.3)
        n, m = npt or 100000, npv or 16384
        times = np.linspace(-0.5, 0.5, n)
        pv = _draw_orbits(rng, m, (0.01, 0.3), 0.7, 0.5)
        ld = _draw_quadratic(rng, m).reshape(m, 1, 2)
        lc, pb, ns, et = _single_lc(n, 3, 2.0 / 1440.0)
        return Workload(name, model, times, lc, pb, ns, et, pv, "quadratic", ld)
    raise ValueError(f"config must be 0..4, got {config}")


def paper_dummy_example() -> dict:
    """The paper's only worked set-up: three light curves, two passbands."""
    return dict(times=np.array([0.0, 1.0, 2.0, 3.0, 4.0, 5.0]),
                lc_index=np.array([0, 0, 1, 1, 1, 2], np.int32),
                passband_index=np.array([0, 1, 0], np.int32))
