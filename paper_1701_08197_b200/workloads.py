"""Seeded synthetic inputs shaped after the paper's four flagger placements (PAPER.md:63-71,
:85, :122-128, :136-138) and BASELINE.json's five configs.  The recipe is stated in DESIGN.md §4.

This module holds NONE of the method's arithmetic (no statistics, thresholds, window sums or
history logic) — it only draws noise, adds rectangles of interference and records where it
put them.  It serves both the oracle-side tests and the CUDA-side tests/bench, and imports
neither.  The paper's recorded observation (pulsar B1919+21) is not available; these inputs
stand in for it.
"""
import math
from dataclasses import dataclass, field

import numpy as np


def _rng(seed, *key):
    """Independent generator per (seed, config, block, stream/station, purpose)."""
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([int(seed)] + [int(k) for k in key])))


def _logu(rng, lo, hi, size=None):
    return np.exp(rng.uniform(math.log(lo), math.log(hi), size))


@dataclass
class Workload:
    name: str
    S: int
    C: int
    T: int
    max_window: int
    block_seconds: float = 1.0
    power: np.ndarray = None          # float32 [S][C][T]  (None for ci16 input)
    volt: np.ndarray = None           # int16 [S][C][T][2] (config 4)
    truth: np.ndarray = None          # uint8 [S][C][T] ground-truth RFI mask, or None
    extra: dict = field(default_factory=dict)

    @property
    def n_samples(self):
        return self.S * self.C * self.T


# ----------------------------------------------------------------------------- config 1
def config1(seed=0):
    """1 x 16 x 256, Exp(1) noise; channel 5 += 20; time 100 += 50; c in [8,16), t in [160,168) += 10."""
    C, T = 16, 256
    x = _rng(seed, 1, 0, 0, 0).standard_exponential((1, C, T)).astype(np.float32)
    truth = np.zeros((1, C, T), np.uint8)
    cls = np.zeros((1, C, T), np.uint8)          # 1 narrowband, 2 broadband spike, 3 burst
    x[0, 5, :] += 20.0; truth[0, 5, :] = 1; cls[0, 5, :] = 1
    x[0, :, 100] += 50.0; truth[0, :, 100] = 1; cls[0, :, 100] = 2
    x[0, 8:16, 160:168] += 10.0; truth[0, 8:16, 160:168] = 1
    cls[0, 8:16, 160:168] = np.where(cls[0, 8:16, 160:168] == 0, 3, cls[0, 8:16, 160:168])
    return Workload("cfg1_tiny", 1, C, T, 32, power=x, truth=truth, extra={"cls": cls})


# ------------------------------------------------------------- shared event model (configs 2, 3)
def _station_events(rng, C, T, spike_rate=5.0, burst_rate=8.0):
    """Rectangles (c0, c1, t0, t1, A): persistent narrowband channels, broadband spikes of
    width 1-4, bursts of 2-128 samples x 1-16 channels; amplitudes log-uniform in [3, 100] sigma."""
    ev = []
    for c in rng.choice(C, size=max(1, round(0.02 * C)), replace=False):
        ev.append((int(c), int(c) + 1, 0, T, float(_logu(rng, 3, 100))))
    for _ in range(rng.poisson(spike_rate)):
        w = int(rng.integers(1, 5)); t0 = int(rng.integers(0, T - w + 1))
        ev.append((0, C, t0, t0 + w, float(_logu(rng, 3, 100))))
    for _ in range(rng.poisson(burst_rate)):
        d = min(T, int(round(float(_logu(rng, 2, 128))))); h = min(C, int(rng.integers(1, 17)))
        t0 = int(rng.integers(0, T - d + 1)); c0 = int(rng.integers(0, C - h + 1))
        ev.append((c0, c0 + h, t0, t0 + d, float(_logu(rng, 3, 100))))
    return ev


def event_class(c0, c1, t0, t1, C, T):
    """Injection class of a rectangle of the shared event model: 1 persistent narrow-band channel (all of time),
    2 broadband spike (all channels), 3 burst."""
    return 1 if (t0 == 0 and t1 == T) else (2 if (c0 == 0 and c1 == C) else 3)


def config2(seed=0, n_subbands=1, n_stations=48, C=64, T=768, want_truth=True):
    """LOFAR-like pre-correlation block: (48 stations x 2 pol) x n_subbands streams of 64 x 768.
    g[c]*Exp(1) with g = 1 + 0.3 sin(2 pi c / C); both polarisations of a station share events."""
    S = n_stations * 2 * n_subbands
    g = (1.0 + 0.3 * np.sin(2 * np.pi * np.arange(C) / C)).astype(np.float32)
    x = np.empty((S, C, T), np.float32)
    truth = np.zeros((S, C, T), np.uint8) if want_truth else None
    cls = np.zeros((S, C, T), np.uint8) if want_truth else None      # 1 narrow-band, 2 spike, 3 burst; amp: its A
    amp = np.zeros((S, C, T), np.float32) if want_truth else None
    for b in range(n_subbands):
        for st in range(n_stations):
            ev = _station_events(_rng(seed, 2, b, st, 1), C, T)
            for pol in range(2):
                s = (b * n_stations + st) * 2 + pol
                xs = _rng(seed, 2, b, s, 0).standard_exponential((C, T), dtype=np.float32)
                xs *= g[:, None]
                for (c0, c1, t0, t1, A) in ev:
                    xs[c0:c1, t0:t1] += np.float32(A)
                    if want_truth:
                        truth[s, c0:c1, t0:t1] = 1
                        k = event_class(c0, c1, t0, t1, C, T)
                        cls[s, c0:c1, t0:t1] = np.maximum(cls[s, c0:c1, t0:t1], k)
                        amp[s, c0:c1, t0:t1] += np.float32(A)
                x[s] = xs
    return Workload(f"cfg2_precorr_x{n_subbands}", S, C, T, 64, power=x, truth=truth,
                    extra={"cls": cls, "amp": amp} if want_truth else {})


def config3(seed=0, n_stations=62, C=16, T=768, max_baselines=None, want_truth=True):
    """Visibility-shaped block: baselines x 4 pol products of 16 x 768; x = |n + sum sqrt(A) e^{i phi}|^2,
    n complex Gaussian with E|n|^2 = 1; baseline (i, j) carries the events of stations i and j."""
    pairs = [(i, j) for i in range(n_stations) for j in range(i + 1, n_stations)]
    if max_baselines is not None:
        pairs = pairs[:max_baselines]
    S = len(pairs) * 4
    events = [_station_events(_rng(seed, 3, 0, st, 1), C, T) for st in range(n_stations)]
    x = np.empty((S, C, T), np.float32)
    truth = np.zeros((S, C, T), np.uint8) if want_truth else None
    cls = np.zeros((S, C, T), np.uint8) if want_truth else None
    for b, (i, j) in enumerate(pairs):
        for pol in range(4):
            s = b * 4 + pol
            r = _rng(seed, 3, 0, s, 0)
            re = r.standard_normal((C, T), dtype=np.float32) * np.float32(math.sqrt(0.5))
            im = r.standard_normal((C, T), dtype=np.float32) * np.float32(math.sqrt(0.5))
            for st in (i, j):
                for e, (c0, c1, t0, t1, A) in enumerate(events[st]):
                    phi = _rng(seed, 3, 0, st, 2, e).uniform(0, 2 * math.pi)
                    re[c0:c1, t0:t1] += np.float32(math.sqrt(A) * math.cos(phi))
                    im[c0:c1, t0:t1] += np.float32(math.sqrt(A) * math.sin(phi))
                    if want_truth:
                        truth[s, c0:c1, t0:t1] = 1
                        cls[s, c0:c1, t0:t1] = np.maximum(cls[s, c0:c1, t0:t1], event_class(c0, c1, t0, t1, C, T))
            x[s] = re * re + im * im
    return Workload("cfg3_visibility", S, C, T, 64, power=x, truth=truth, extra={"cls": cls} if want_truth else {})


# ----------------------------------------------------------------------------- config 4
def config4(seed=0, n_stations=48, C=32, T=195312, want_truth=False):
    """Raw-voltage high-time-resolution block: (48 x 2) streams x 32 subbands x 195 312 samples of
    complex int16, re, im = round(N(0, 32^2)).  Spikes: Poisson(200)/s of 1-16 samples over all
    subbands, voltage amplitude log-U[3, 30] x 32; bursts: Poisson(10)/s of 1-10 ms x 1-4 subbands,
    amplitude log-U[1.5, 10] x 32; clipped to int16.  Rates scale with T / 195312."""
    S = n_stations * 2
    sec = T / 195312.0
    v = np.empty((S, C, T, 2), np.int16)
    truth = np.zeros((S, C, T), np.uint8) if want_truth else None
    cls = np.zeros((S, C, T), np.uint8) if want_truth else None       # 2 spike (all subbands), 3 burst
    for st in range(n_stations):
        r = _rng(seed, 4, 0, st, 1)
        ev = []
        for _ in range(r.poisson(200.0 * sec)):
            w = int(r.integers(1, 17)); t0 = int(r.integers(0, max(1, T - w + 1)))
            ev.append((0, C, t0, min(T, t0 + w), 32.0 * float(_logu(r, 3, 30)), float(r.uniform(0, 2 * math.pi))))
        for _ in range(r.poisson(10.0 * sec)):
            d = min(T, int(r.integers(195, 1954))); h = int(r.integers(1, 5))
            t0 = int(r.integers(0, T - d + 1)); c0 = int(r.integers(0, C - h + 1))
            ev.append((c0, c0 + h, t0, t0 + d, 32.0 * float(_logu(r, 1.5, 10)), float(r.uniform(0, 2 * math.pi))))
        for pol in range(2):
            s = st * 2 + pol
            f = _rng(seed, 4, 0, s, 0).standard_normal((C, T, 2), dtype=np.float32)
            f *= np.float32(32.0)
            for (c0, c1, t0, t1, A, phi) in ev:
                f[c0:c1, t0:t1, 0] += np.float32(A * math.cos(phi))
                f[c0:c1, t0:t1, 1] += np.float32(A * math.sin(phi))
                if want_truth:
                    truth[s, c0:c1, t0:t1] = 1
                    cls[s, c0:c1, t0:t1] = np.maximum(cls[s, c0:c1, t0:t1], 2 if (c0 == 0 and c1 == C) else 3)
            np.rint(f, out=f)
            np.clip(f, -32768, 32767, out=f)
            v[s] = f.astype(np.int16)
    return Workload("cfg4_rawvoltage", S, C, T, 256, volt=v, truth=truth, extra={"cls": cls} if want_truth else {})


# ----------------------------------------------------------------------------- config 5
class Config5Stream:
    """Beam-formed Stokes-I stream of blocks: 488 subbands x 16 channels x 12 208 samples (81.92 us),
    chi^2_4 / 4 noise (mean 1, sigma 0.7071) x a bandpass drifting by a factor (1+u), u~U[-0.05,0.05]
    per (s, c) per block; 2 % of rows carry narrowband RFI switching on/off between blocks
    (P(switch) = 0.3), amplitude log-U[3, 100] sigma; plus a dispersed periodic pulse (period
    1.3373 s, width 0.04 s, DM 12.455 over 138.0-145.2 MHz) of +0.5 sigma that is
    NOT in the ground-truth mask."""

    SIGMA = math.sqrt(0.5)

    def __init__(self, seed=0, S=488, C=16, T=12208, want_truth=True):
        self.seed, self.S, self.C, self.T, self.want_truth = seed, S, C, T, want_truth
        self.k = 0
        self.band = np.ones((S, C), np.float64)
        r = _rng(seed, 5, 0, 0, 1)
        rows = S * C
        self.rfi_rows = r.choice(rows, size=max(1, round(0.02 * rows)), replace=False)
        self.rfi_amp = _logu(r, 3, 100, self.rfi_rows.size) * self.SIGMA
        self.rfi_on = r.random(self.rfi_rows.size) < 0.5
        # frequency of row (s, c): 138.0 .. 145.2 MHz, lowest first
        f = 138.0 + (145.2 - 138.0) * (np.arange(rows) + 0.5) / rows
        self.delay = 4.148808e3 * 12.455 * (f ** -2 - 145.2 ** -2)        # seconds (cold-plasma delay)
        self.dt = 1.0 / T

    def next_block(self):
        S, C, T, k = self.S, self.C, self.T, self.k
        if k > 0:
            rb = _rng(self.seed, 5, k, 0, 2)
            self.band *= 1.0 + rb.uniform(-0.05, 0.05, (S, C))
            flip = _rng(self.seed, 5, k, 0, 3).random(self.rfi_rows.size) < 0.3
            self.rfi_on = np.logical_xor(self.rfi_on, flip)
        x = np.empty((S, C, T), np.float32)
        for s in range(S):
            xs = _rng(self.seed, 5, k, s, 0).standard_gamma(2.0, (C, T), dtype=np.float32)
            xs *= np.float32(0.5)
            x[s] = xs
        # dispersed pulse: additive 0.5 sigma where ((t_abs - delay) mod period) < width
        t_abs = k * 1.0 + (np.arange(T) + 0.5) * self.dt
        pulse = np.zeros((S * C, T), np.uint8)
        for r_ in range(S * C):
            ph = np.mod(t_abs - self.delay[r_], 1.3373)
            pulse[r_] = ph < 0.04
        x2 = x.reshape(S * C, T)
        x2 += pulse.astype(np.float32) * np.float32(0.5 * self.SIGMA)
        truth = np.zeros((S * C, T), np.uint8) if self.want_truth else None
        on_rows = self.rfi_rows[self.rfi_on]
        x2[on_rows] += self.rfi_amp[self.rfi_on].astype(np.float32)[:, None]
        if truth is not None:
            truth[on_rows] = 1
        x2 *= self.band.reshape(S * C, 1).astype(np.float32)
        self.k += 1
        return Workload(f"cfg5_beamformed_block{k}", S, C, T, 64, power=x,
                        truth=None if truth is None else truth.reshape(S, C, T),
                        extra={"pulse": pulse.reshape(S, C, T), "rfi_rows_on": on_rows,
                               "band": self.band.copy()})


def tile_streams(w, factor):
    """Repeat a workload's streams `factor` times with a per-copy time roll (keeps value
    distribution and RFI structure; used to reach bench sizes larger than L2 quickly)."""
    parts, truths = [], []
    src = w.power if w.power is not None else w.volt
    for i in range(factor):
        parts.append(np.roll(src, 37 * i, axis=2))
        if w.truth is not None:
            truths.append(np.roll(w.truth, 37 * i, axis=2))
    big = np.concatenate(parts, axis=0)
    out = Workload(f"{w.name}_tiled{factor}", w.S * factor, w.C, w.T, w.max_window, w.block_seconds,
                   truth=np.concatenate(truths, axis=0) if truths else None)
    if w.power is not None:
        out.power = big
    else:
        out.volt = big
    return out
