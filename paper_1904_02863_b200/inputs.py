"""Seeded synthetic inputs for the five BASELINE.json workloads (C0..C4).

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench.  It
holds none of the method's arithmetic: no waveform, no antenna pattern, no inner
product.  The injection needs a waveform, so ``make_data`` takes it as a callable
(the tests pass the oracle's; ``bench.py`` passes the library's own
``gw_waveform_batch``).  Recipe: SURVEY.md 8(d) "Synthetic inputs", restated in
DESIGN.md section 4; shapes from BASELINE.json ``configs[0..4]``.

The paper measures on simulated signals of a given duration in Gaussian noise
(PAPER.md:47 durations, PAPER.md:67 bin counts, PAPER.md:75-81 synthetic BNS);
no public dataset is involved, these inputs stand in for its duration sweep.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Callable, Optional, Tuple

import numpy as np

BASE_SEED = 19040286

# theta column order == GW_P_* enum of include/gwlnl.h
P_MC, P_Q, P_CHI1, P_CHI2, P_DL, P_TC, P_PHIC, P_COSI, P_RA, P_DEC, P_PSI = range(11)
NPARAM = 11
DET_ROW = 13  # kind, vertex[3], xarm[3], yarm[3], fplus, fcross, dt

# "standard H1/L1/V1 vertex and arm geometry" (BASELINE.json configs[1]); digits as listed in
# SURVEY.md 8(c); input data, pinned by invariants only (tests/test_inputs.py).
_GEOMETRY = {
    "H1": ((-2.16141492636e6, -3.83469517889e6, 4.60035022664e6),
           (-0.22389266154, 0.79983062746, 0.55690487831),
           (-0.91397818574, 0.02609403989, -0.40492342125)),
    "L1": ((-7.42760447238e4, -5.49628371971e6, 3.22425701744e6),
           (-0.95457412153, -0.14158077340, -0.26218911324),
           (0.29774156894, -0.48791033647, -0.82054461286)),
    "V1": ((4.54637409900e6, 8.42989697626e5, 4.37857696241e6),
           (-0.70045821479, 0.20848948619, 0.68256166277),
           (-0.05379255368, -0.96908180549, 0.24080451708)),
}


def geometric_detector(name: str) -> np.ndarray:
    r, x, y = _GEOMETRY[name]
    row = np.zeros(DET_ROW)
    row[0] = 0.0
    row[1:4], row[4:7], row[7:10] = r, x, y
    return row


def fixed_detector(fplus: float, fcross: float, dt_s: float) -> np.ndarray:
    row = np.zeros(DET_ROW)
    row[0] = 1.0
    row[10], row[11], row[12] = fplus, fcross, dt_s
    return row


@dataclass(frozen=True)
class Config:
    """One BASELINE.json workload.  ``index`` is the 0-based position in ``configs``."""
    name: str
    index: int
    det_names: Tuple[str, ...]          # () => one FIXED detector (F+=1, Fx=0, dt=0)
    duration_s: float                   # T; delta_f = 1/T
    f_min: float
    f_max: float
    batch: int
    mc_range: Tuple[float, float]
    q_range: Tuple[float, float]
    dl_range: Tuple[float, float]
    chi_range: Tuple[float, float]      # (0,0) => non-spinning
    theta_inj: Tuple[float, ...]        # 11 values, GW_P_* order
    gmst: float = 2.0
    spin_order: int = 1

    @property
    def n_det(self) -> int:
        return max(1, len(self.det_names))

    @property
    def delta_f(self) -> float:
        return 1.0 / self.duration_s

    @property
    def n_bins(self) -> int:
        return int(round((self.f_max - self.f_min) * self.duration_s)) + 1

    @property
    def seed_noise(self) -> int:
        return BASE_SEED + 10 * self.index + 1

    @property
    def seed_prop(self) -> int:
        return BASE_SEED + 10 * self.index + 2

    def reduced(self, *, f_max: Optional[float] = None, batch: Optional[int] = None,
                duration_s: Optional[float] = None) -> "Config":
        """Same recipe and seeds on a narrower band / smaller batch / shorter segment (test sizes)."""
        return replace(self, f_max=self.f_max if f_max is None else f_max,
                       batch=self.batch if batch is None else batch,
                       duration_s=self.duration_s if duration_s is None else duration_s)


_INJ_BBH0 = (28.0, 0.8, 0.0, 0.0, 500.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0)
_INJ_BBH = (28.0, 0.8, 0.3, -0.2, 500.0, 0.01, 1.3, 0.8, 1.0, -0.5, 0.7)
_INJ_BNS = (1.2, 0.9, 0.02, -0.01, 100.0, 0.01, 1.3, 0.8, 1.0, -0.5, 0.7)
_HLV = ("H1", "L1", "V1")

CONFIGS = {
    "C0": Config("C0", 0, (), 8.0, 20.0, 512.0, 256, (20, 40), (0.5, 1), (200, 2000), (0, 0),
                 _INJ_BBH0, spin_order=0),
    "C1": Config("C1", 1, _HLV, 4.0, 20.0, 2048.0, 4096, (20, 40), (0.5, 1), (200, 2000), (-0.8, 0.8),
                 _INJ_BBH),
    "C2": Config("C2", 2, _HLV, 128.0, 20.0, 2048.0, 1024, (1.1, 1.3), (0.7, 1), (20, 200), (-0.05, 0.05),
                 _INJ_BNS),
    "C3": Config("C3", 3, _HLV, 512.0, 10.0, 2048.0, 256, (1.1, 1.3), (0.7, 1), (20, 200), (-0.05, 0.05),
                 _INJ_BNS),
    "C4": Config("C4", 4, _HLV, 4.0, 20.0, 2048.0, 65536, (20, 40), (0.5, 1), (200, 2000), (-0.8, 0.8),
                 _INJ_BBH),
}
C4_BATCHES = (1, 16, 256, 4096, 65536)


def frequency_grid(cfg: Config) -> np.ndarray:
    """f_j = f_min + j*delta_f, j = 0..M-1 (both band edges included)."""
    return cfg.f_min + np.arange(cfg.n_bins, dtype=np.float64) * cfg.delta_f


def analytic_psd(freqs: np.ndarray) -> np.ndarray:
    """S_n(f) = 1e-49 [x^-4.14 - 5 x^-2 + 111 (1 - x^2 + x^4/2)/(1 + x^2/2)], x = f/215 Hz
    (BASELINE.json configs[0]); one-sided, strain^2/Hz, positive on [10, 2048] Hz."""
    x = np.asarray(freqs, dtype=np.float64) / 215.0
    x2 = x * x
    return 1e-49 * (x ** -4.14 - 5.0 / x2 + 111.0 * (1.0 - x2 + 0.5 * x2 * x2) / (1.0 + 0.5 * x2))


def detectors(cfg: Config) -> np.ndarray:
    """[n_det][13] rows (see DET_ROW)."""
    if not cfg.det_names:
        return fixed_detector(1.0, 0.0, 0.0)[None, :]
    return np.stack([geometric_detector(n) for n in cfg.det_names])


def psd(cfg: Config) -> np.ndarray:
    """[n_det][M]: the same analytic PSD for every detector."""
    return np.tile(analytic_psd(frequency_grid(cfg)), (cfg.n_det, 1))


def proposals(cfg: Config, batch: Optional[int] = None) -> np.ndarray:
    """theta[B][11]: u = rng.random((B_cfg, 11)) mapped affinely, row 0 := theta_inj.
    A smaller ``batch`` is a prefix of the config's draw (C4 sweep)."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed_prop))
    u = rng.random((cfg.batch, NPARAM))

    def lin(col, lo, hi):
        return lo + (hi - lo) * u[:, col]

    th = np.empty_like(u)
    th[:, P_MC] = lin(P_MC, *cfg.mc_range)
    th[:, P_Q] = lin(P_Q, *cfg.q_range)
    th[:, P_CHI1] = lin(P_CHI1, *cfg.chi_range)
    th[:, P_CHI2] = lin(P_CHI2, *cfg.chi_range)
    th[:, P_DL] = lin(P_DL, *cfg.dl_range)
    th[:, P_TC] = lin(P_TC, -0.1, 0.1)
    th[:, P_PHIC] = lin(P_PHIC, 0.0, 2.0 * np.pi)
    if cfg.det_names:
        th[:, P_COSI] = 2.0 * u[:, P_COSI] - 1.0
        th[:, P_RA] = 2.0 * np.pi * u[:, P_RA]
        th[:, P_DEC] = np.arcsin(2.0 * u[:, P_DEC] - 1.0)
        th[:, P_PSI] = np.pi * u[:, P_PSI]
    else:  # C0: optimally oriented, fixed response
        th[:, P_COSI] = 1.0
        th[:, P_RA] = th[:, P_DEC] = th[:, P_PSI] = 0.0
    th[0, :] = cfg.theta_inj
    if batch is not None:
        if batch > cfg.batch:
            raise ValueError("batch larger than the config's draw")
        th = th[:batch]
    return np.ascontiguousarray(th)


def tidal_lambdas(cfg: Config, batch: Optional[int] = None, lam_max: float = 5000.0) -> np.ndarray:
    """lambdas[B][2]: dimensionless tidal deformabilities (Lambda_1, Lambda_2) ~ U[0, lam_max] for the tidal option
    (NEXT-1; the usual prior range of neutron-star analyses), drawn from a stream of their own so that the
    11-column proposals above are unchanged.  Row 0 (the injection's slot) is (400, 600)."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed_prop + 5))
    lam = lam_max * rng.random((cfg.batch, 2))
    lam[0, :] = (400.0, 600.0)
    return np.ascontiguousarray(lam if batch is None else lam[:batch])


def noise(cfg: Config) -> np.ndarray:
    """n[n_det][M] complex: Re and Im each N(0, S/(4 delta_f)), independent per detector and bin."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed_noise))
    z = rng.standard_normal((cfg.n_det, cfg.n_bins, 2))
    sigma = np.sqrt(psd(cfg) / (4.0 * cfg.delta_f))
    return (z[..., 0] + 1j * z[..., 1]) * sigma


WaveformFn = Callable[[np.ndarray, np.ndarray, float, np.ndarray, int], np.ndarray]


def make_data(cfg: Config, waveform_fn: WaveformFn) -> np.ndarray:
    """d[n_det][M] = injection + noise.  ``waveform_fn(freqs, dets, gmst, theta[1][11], spin_order)``
    must return h[1][n_det][M] complex128; this module does not know how."""
    th = np.asarray(cfg.theta_inj, dtype=np.float64)[None, :]
    s = np.asarray(waveform_fn(frequency_grid(cfg), detectors(cfg), cfg.gmst, th, cfg.spin_order))
    return s.reshape(cfg.n_det, cfg.n_bins) + noise(cfg)


# ---- population likelihood workloads (section IV, Eq. 3) --------------------------
# Synthetic posterior samples stand in for the GWTC-1 release the paper used (ten events, >= 2e4 samples
# each) and for its projected catalogues (up to ~4e6 samples); nothing here evaluates a population model.
POP_NTHETA = 6       # m1 [Msun], q, a1, a2, cos tilt1, cos tilt2
POP_NLAMBDA = 12     # alpha, m_min, m_max, lam, m_pp, sig_pp, beta_q, alpha_chi, beta_chi, xi, sig_1, sig_2
POP_M1_RANGE = (2.5, 95.0)


@dataclass(frozen=True)
class PopConfig:
    name: str
    index: int
    n_events: int
    n_samples: int
    batch: int           # hyper-parameter proposals Lambda per call

    @property
    def seed_samples(self) -> int:
        return BASE_SEED + 100 + 10 * self.index + 1

    @property
    def seed_prop(self) -> int:
        return BASE_SEED + 100 + 10 * self.index + 2


POP_CONFIGS = {
    "P0": PopConfig("P0", 0, 10, 2000, 64),        # small: the oracle finishes in seconds
    "P1": PopConfig("P1", 1, 10, 20000, 64),       # 2e5 samples: the size of the GWTC-1 release
    "P2": PopConfig("P2", 2, 100, 40000, 64),      # 4e6 samples: where the paper's P100 saturates
}


def pop_samples(cfg: PopConfig) -> Tuple[np.ndarray, np.ndarray]:
    """(samples [N][n][6], prior [N][n]): per event a Gaussian cloud around a random centre, folded into the domain;
    the prior the clouds are weighted by is p(theta | 0) = (2 m1 / (hi^2 - lo^2)) * 1 * 1 * 1 * (1/4) -- flat in the
    component masses, in both spin magnitudes and in both tilt cosines."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed_samples))
    N, n = cfg.n_events, cfg.n_samples
    lo = np.array([POP_M1_RANGE[0], 0.05, 0.005, 0.005, -0.999, -0.999])
    hi = np.array([POP_M1_RANGE[1], 1.0, 0.995, 0.995, 0.999, 0.999])
    c_lo = np.array([8.0, 0.5, 0.05, 0.05, -0.5, -0.5])
    c_hi = np.array([45.0, 0.95, 0.6, 0.6, 0.9, 0.9])
    centre = c_lo + (c_hi - c_lo) * rng.random((N, POP_NTHETA))
    width = np.array([0.0, 0.12, 0.15, 0.15, 0.35, 0.35]) + np.zeros((N, POP_NTHETA))
    width[:, 0] = 0.1 * centre[:, 0]
    x = centre[:, None, :] + width[:, None, :] * rng.standard_normal((N, n, POP_NTHETA))
    span = hi - lo                                      # fold into [lo, hi] by reflection
    y = np.mod(x - lo, 2.0 * span)
    x = lo + np.where(y > span, 2.0 * span - y, y)
    prior = 2.0 * x[..., 0] / (POP_M1_RANGE[1] ** 2 - POP_M1_RANGE[0] ** 2) * 0.25
    return np.ascontiguousarray(x), np.ascontiguousarray(prior)


def pop_lambdas(cfg: PopConfig, batch: Optional[int] = None) -> np.ndarray:
    """Lambda[B][12] drawn uniformly from the usual prior ranges of a population analysis; row 0 is a fixed, typical
    point.  (beta_q stays away from -1 and alpha from 1, the two removable singularities of the normalisations.)"""
    rng = np.random.Generator(np.random.PCG64(cfg.seed_prop))
    lo = np.array([1.2, 3.0, 50.0, 0.0, 25.0, 1.0, -0.5, 1.0, 1.0, 0.0, 0.3, 0.3])
    hi = np.array([4.0, 8.0, 90.0, 0.3, 40.0, 8.0, 4.0, 5.0, 6.0, 1.0, 3.0, 3.0])
    lam = lo + (hi - lo) * rng.random((cfg.batch, POP_NLAMBDA))
    lam[0] = (2.35, 5.0, 70.0, 0.1, 33.0, 5.0, 1.3, 2.0, 4.0, 0.6, 1.0, 1.5)
    return np.ascontiguousarray(lam if batch is None else lam[:batch])
