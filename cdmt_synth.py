"""Seeded synthetic complex-voltage inputs for the five BASELINE.json configs.

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU
oracle's tests.  It holds no step of the cdmt method (no segmenting, no
channelising, no detection): it only synthesises *telescope-like input*, i.e.
dual-polarisation Nyquist-sampled complex voltages per subband
(PAPER.md:77, 137), with noise plus test signals that have been *dispersed*
the way the interstellar medium would (the conjugate of PAPER.md:57 Eq. 1, typed
here independently in numpy so that a mistake in either the oracle's or the
kernels' chirp shows up as a pulse recovered at the wrong DM).

The recordings the paper used (LOFAR HBA, 200 x 195.3125 kHz subbands at
135 MHz, int8) are not available; these inputs stand in for
them with the same shapes, word sizes, sampling (5.12 us) and DM ranges.

Layout of every array returned: ``[2 pols][T samples]`` complex64, or
``[2][T][2]`` int8 (re, im interleaved) for the int8 config; a whole config is
``[nsub][2][T]`` in ascending subband frequency.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

BW_MHZ = 0.1953125            # LOFAR subband width = complex sample rate
TSAMP_S = 1.0 / (BW_MHZ * 1e6)  # 5.12 us
KDM_INV = 2.41e-4             # k_DM^-1 in s MHz^2

REF_CHANNEL = 0
REF_SUBBAND = 1
IN_CF32 = 0
IN_CI8 = 1


@dataclass
class Impulse:
    n0: int          # arrival sample (input samples) at the reference frequency
    amp: float       # amplitude A of the undispersed delta
    dm: float        # DM it is dispersed with


@dataclass
class Config:
    name: str
    nsub: int
    fcen_mhz: np.ndarray          # [nsub] ascending
    nsamp: int                    # T, samples per pol per subband
    nfft: int
    noverlap: int
    nchan: int
    ndec: int
    dm: np.ndarray                # [ndm]
    seed: int
    in_dtype: int = IN_CF32
    bw_mhz: float = BW_MHZ
    noise_sigma: float = 1.0      # per complex sample: E|x|^2 = sigma^2 (cf32) ; per component for int8
    impulses: List[Impulse] = field(default_factory=list)
    pulse_train: Optional[Tuple[float, float, float, float]] = None  # (period_samples, duty, amp, dm)

    # derived sizes (bookkeeping of PAPER.md:81, 113, 123; no arithmetic of the method)
    @property
    def ndm(self) -> int:
        return int(self.dm.size)

    @property
    def step(self) -> int:
        return self.nfft - self.noverlap

    @property
    def nblock(self) -> int:
        return (self.nsamp - self.nfft) // self.step + 1

    @property
    def mbin(self) -> int:
        return self.nfft // self.nchan

    @property
    def half_discard(self) -> int:
        return self.noverlap // (2 * self.nchan)

    @property
    def nvalid_dec(self) -> int:
        return (self.mbin - 2 * self.half_discard) // self.ndec

    def plan_kwargs(self, chirp_ref: int = REF_CHANNEL) -> dict:
        return dict(nsub=self.nsub, fcen_mhz=self.fcen_mhz, bw_mhz=self.bw_mhz,
                    nfft=self.nfft, noverlap=self.noverlap, nchan=self.nchan,
                    ndec=self.ndec, dm=self.dm, in_dtype=self.in_dtype,
                    chirp_ref=chirp_ref)


def _contig_fcen(f_lo_mhz: float, nsub: int) -> np.ndarray:
    return f_lo_mhz + (np.arange(nsub) + 0.5) * BW_MHZ


def make_config(name: str) -> Config:
    """The five workloads of BASELINE.json `configs` (recipe: SURVEY.md 8(d) table)."""
    if name in ("c1", "tiny"):
        cfg = Config("c1", 1, np.array([150.0]), 2 ** 14, 4096, 1024, 8, 4,
                     np.array([0.0, 2.0, 4.0, 6.0]), seed=0)
        cfg.impulses = [Impulse(n0=7008, amp=50.0, dm=4.0)]
        return cfg
    if name == "c2":
        cfg = Config("c2", 20, _contig_fcen(130.0, 20), 2 ** 20, 65536, 8192, 8, 8,
                     0.3125 * np.arange(128), seed=1)
        rng = np.random.default_rng([cfg.seed, 10 ** 6])
        C, D = cfg.nchan, cfg.ndec
        for _ in range(5):
            dm = float(rng.uniform(0.0, 40.0))
            n0 = int(rng.integers(cfg.nfft, cfg.nsamp - cfg.nfft)) // C * C
            snr = float(rng.uniform(8.0, 20.0))
            amp = float(np.sqrt(snr * C * np.sqrt(2.0 * D) / 2.0))
            cfg.impulses.append(Impulse(n0, amp, dm))
        return cfg
    if name == "c3":
        cfg = Config("c3", 288, _contig_fcen(119.0, 288), 2 ** 21, 65536, 16384, 16, 16,
                     0.5 * np.arange(96), seed=2)
        cfg.pulse_train = (3.1e-3 / TSAMP_S, 0.05, 1.0, 21.0)
        return cfg
    if name == "c4":
        fc = 135.0 + (np.arange(64) - 31.5) * BW_MHZ
        cfg = Config("c4", 64, fc, 2 ** 22, 262144, 131072, 32, 32,
                     5.0 * np.arange(200), seed=3)
        CD = cfg.nchan * cfg.ndec
        for frac, dm in ((0.25, 250.0), (0.5, 600.0), (0.75, 950.0)):
            cfg.impulses.append(Impulse(int(frac * cfg.nsamp) // CD * CD, 50.0, dm))
        return cfg
    if name == "c5":
        cfg = Config("c5", 64, _contig_fcen(140.0, 64), 2 ** 22, 65536, 32768, 8, 8,
                     0.1 * np.arange(1024), seed=4, in_dtype=IN_CI8, noise_sigma=20.0)
        rng = np.random.default_rng([cfg.seed, 10 ** 6])
        for _ in range(10):
            dm = float(rng.uniform(0.0, 100.0))
            n0 = int(rng.integers(cfg.nfft, cfg.nsamp - cfg.nfft)) // cfg.nchan * cfg.nchan
            cfg.impulses.append(Impulse(n0, 15.0 * cfg.noise_sigma, dm))
        return cfg
    raise KeyError(name)


CONFIG_NAMES = ("c1", "c2", "c3", "c4", "c5")


def small_config(nsub=2, nsamp=4096, nfft=1024, noverlap=256, nchan=4, ndec=2,
                 dm=(0.0, 1.5, 3.0), f_lo=140.0, seed=7, in_dtype=IN_CF32,
                 name="small") -> Config:
    """A free-form small workload for tests (same recipe: unit noise, no injected signal)."""
    sigma = 20.0 if in_dtype == IN_CI8 else 1.0
    return Config(name, nsub, _contig_fcen(f_lo, nsub), nsamp, nfft, noverlap, nchan, ndec,
                  np.asarray(dm, dtype=np.float64), seed=seed, in_dtype=in_dtype,
                  noise_sigma=sigma)


# ---------------------------------------------------------------------------
# ISM dispersion of a test signal (conjugate of PAPER.md:57 Eq. 1), numpy, fp64.
# ---------------------------------------------------------------------------

def ism_phase_cycles(dm: float, f0_mhz, f_off_mhz):
    """Phase of Eq. 1 in cycles: DM f^2 / (2.41e-10 f0^2 (f0+f)), f, f0 in MHz."""
    f0 = np.asarray(f0_mhz, dtype=np.float64)
    f = np.asarray(f_off_mhz, dtype=np.float64)
    return dm * f * f / (KDM_INV * 1e-6 * f0 * f0 * (f0 + f))


def _bin_offsets_mhz(T: int, bw_mhz: float) -> np.ndarray:
    """Frequency offset from the subband centre of numpy-FFT bin k of a length-T transform."""
    k = np.arange(T)
    k = np.where(k < T // 2, k, k - T)       # bins T/2.. are negative frequencies
    return k * (bw_mhz / T)


def disperse(sig: np.ndarray, dm: float, fcen_mhz: float, bw_mhz: float, nchan: int,
             chirp_ref: int) -> np.ndarray:
    """Circularly convolve `sig` (complex, length T) with the ISM response at `dm`.

    chirp_ref=REF_SUBBAND: one chirp over the subband, referenced to its centre.
    chirp_ref=REF_CHANNEL: each of the `nchan` equal channels gets the chirp referenced
    to its own centre (so that a plan in the same mode recovers the pulse at one sample
    in every channel)."""
    T = sig.size
    spec = np.fft.fft(sig.astype(np.complex128))
    f = _bin_offsets_mhz(T, bw_mhz)
    if chirp_ref == REF_SUBBAND:
        ph = ism_phase_cycles(dm, fcen_mhz, f)
    else:
        cw = bw_mhz / nchan
        c = np.floor((f + bw_mhz / 2.0) / cw)
        c = np.clip(c, 0, nchan - 1)
        fc_off = (c + 0.5) * cw - bw_mhz / 2.0        # channel centre offset from subband centre
        ph = ism_phase_cycles(dm, fcen_mhz + fc_off, f - fc_off)
    ph -= np.rint(ph)
    spec *= np.exp(-2j * np.pi * ph)                  # conjugate of Eq. 1: the ISM, not its removal
    return np.fft.ifft(spec)


def _signal_for_subband(cfg: Config, s: int, chirp_ref: int) -> Optional[np.ndarray]:
    T = cfg.nsamp
    total = None
    by_dm = {}
    for imp in cfg.impulses:
        d = by_dm.setdefault(imp.dm, np.zeros(T, dtype=np.complex128))
        d[imp.n0] += imp.amp
    if cfg.pulse_train is not None:
        period, duty, amp, dm = cfg.pulse_train
        rng = np.random.default_rng([cfg.seed, 2 * 10 ** 6, s])
        n = np.arange(T)
        on = np.mod(n, period) < duty * period
        g = (rng.standard_normal(T) + 1j * rng.standard_normal(T)) / np.sqrt(2.0)
        d = by_dm.setdefault(dm, np.zeros(T, dtype=np.complex128))
        d += amp * g * on
    for dm, d in by_dm.items():
        y = disperse(d, dm, float(cfg.fcen_mhz[s]), cfg.bw_mhz, cfg.nchan, chirp_ref)
        total = y if total is None else total + y
    return total


def generate_subband(cfg: Config, s: int, chirp_ref: int = REF_CHANNEL) -> np.ndarray:
    """Voltages of subband `s`: [2][T] complex64, or [2][T][2] int8 for IN_CI8."""
    T = cfg.nsamp
    rng = np.random.default_rng([cfg.seed, s])
    sig = _signal_for_subband(cfg, s, chirp_ref)
    if cfg.in_dtype == IN_CF32:
        out = np.empty((2, T), dtype=np.complex64)
        for p in range(2):
            re = rng.standard_normal(T)
            im = rng.standard_normal(T)
            x = (re + 1j * im) * (cfg.noise_sigma / np.sqrt(2.0))
            if sig is not None:
                x = x + sig
            out[p] = x.astype(np.complex64)
        return out
    out = np.empty((2, T, 2), dtype=np.int8)
    for p in range(2):
        re = rng.standard_normal(T) * cfg.noise_sigma
        im = rng.standard_normal(T) * cfg.noise_sigma
        if sig is not None:
            re = re + sig.real
            im = im + sig.imag
        out[p, :, 0] = np.clip(np.rint(re), -127, 127).astype(np.int8)
        out[p, :, 1] = np.clip(np.rint(im), -127, 127).astype(np.int8)
    return out


def generate(cfg: Config, chirp_ref: int = REF_CHANNEL,
             subbands: Optional[Sequence[int]] = None, threads: int = 1) -> np.ndarray:
    """All (or the listed) subbands stacked: [nsub][2][T] complex64 / [nsub][2][T][2] int8."""
    subs = list(range(cfg.nsub)) if subbands is None else list(subbands)
    if threads > 1 and len(subs) > 1:
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(threads) as ex:
            parts = list(ex.map(lambda s: generate_subband(cfg, s, chirp_ref), subs))
    else:
        parts = [generate_subband(cfg, s, chirp_ref) for s in subs]
    return np.stack(parts, axis=0)
