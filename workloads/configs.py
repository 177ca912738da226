"""The five BASELINE.json configurations and their seeded generators.

The dispersion sweep used to *inject* synthetic pulses below is the cold-plasma law
 evaluated for the pulse's own (possibly off-grid) DM: it is a property
of the simulated sky signal, not a piece of the pipeline.  Neither the oracle nor the
CUDA library imports it for their delay tables.
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np

KDM = 4.148808e3  # s MHz^2 pc^-1 cm^3 (north_star)


@dataclass(frozen=True)
class Config:
    name: str
    nbeams: int
    nchans: int
    f_top: float
    foff: float
    tsamp: float
    nsamps: int
    dm_low: float
    dm_step: float
    ndms: int
    dtype: str           # "f32" | "u8"
    seed: int            # beam b uses seed + b
    recipe: str          # "cfg1" | "cfg2" | "cfg4" | "cfg5"
    snr_thresh: float = 6.0
    window: int = 64
    k_chan: float = 5.0
    k_spec: float = 5.0

    @property
    def np_dtype(self):
        return np.float32 if self.dtype == "f32" else np.uint8

    def plan_args(self):
        return (self.nbeams, self.nchans, self.f_top, self.foff, self.tsamp, self.nsamps,
                self.dm_low, self.dm_step, self.ndms)

    def sweep(self, dm: float) -> np.ndarray:
        """Arrival delay in samples of a pulse of dispersion measure `dm` in every channel."""
        f = self.f_top + np.arange(self.nchans, dtype=np.float64) * self.foff
        return np.floor(KDM * dm * (f ** -2.0 - self.f_top ** -2.0) / self.tsamp + 0.5).astype(np.int64)

    @property
    def dm_max(self) -> float:
        return self.dm_low + (self.ndms - 1) * self.dm_step

    @property
    def sweep_max(self) -> int:
        return int(self.sweep(self.dm_max)[-1])


CONFIGS = {
    1: Config("cfg1-tiny", 1, 64, 418.0, -0.3125, 51.2e-6, 4096, 0.0, 0.1, 32, "f32", 1, "cfg1"),
    2: Config("cfg2-one-beam", 1, 1024, 418.0, -0.01953125, 51.2e-6, 65536, 0.0, 0.1, 640, "f32", 2, "cfg2"),
    3: Config("cfg3-8beam-f32", 8, 1024, 418.0, -0.01953125, 51.2e-6, 65536, 0.0, 0.1, 640, "f32", 300, "cfg2"),
    4: Config("cfg4-8beam-u8", 8, 1024, 418.0, -0.01953125, 51.2e-6, 65536, 0.0, 0.1, 640, "u8", 400, "cfg4"),
    5: Config("cfg5-stress", 16, 4096, 418.0, -20.0 / 4096, 51.2e-6, 131072, 0.0, 0.1, 2048, "f32", 500, "cfg5"),
}


def _noise(rng_seed: int, nchans: int, nsamps: int, nthreads: int = 8) -> np.ndarray:
    """N(0,1) float32 [nchans][nsamps]; channel blocks drawn from independent spawned streams
    so the result does not depend on the thread count."""
    out = np.empty((nchans, nsamps), dtype=np.float32)
    blk = 64
    nblk = (nchans + blk - 1) // blk
    seeds = np.random.SeedSequence(rng_seed).spawn(nblk)

    def fill(i):
        g = np.random.Generator(np.random.PCG64(seeds[i]))
        lo, hi = i * blk, min(nchans, (i + 1) * blk)
        g.standard_normal(out=out[lo:hi], dtype=np.float32)

    if nchans * nsamps < (1 << 22):
        for i in range(nblk):
            fill(i)
    else:
        with ThreadPoolExecutor(nthreads) as ex:
            list(ex.map(fill, range(nblk)))
    return out


def _inject(x: np.ndarray, cfg: Config, dm: float, t0: int, width: int, amp) -> None:
    """x[c][t0 + sweep(dm)[c] + i] += amp[c] for i < width, skipped where out of range."""
    sw = cfg.sweep(dm)
    amp = np.broadcast_to(np.asarray(amp, dtype=x.dtype), (cfg.nchans,))
    for c in range(cfg.nchans):
        a = t0 + int(sw[c])
        b = min(a + width, cfg.nsamps)
        if a < cfg.nsamps and b > max(a, 0):
            x[c, max(a, 0):b] += amp[c]


def pulses(cfg: Config, b: int):
    """The list of injected pulses (dm, t0, width, amplitude) of beam b -- a pure function of the seed."""
    g = np.random.Generator(np.random.PCG64(np.random.SeedSequence([cfg.seed + b, 7])))
    nso = cfg.nsamps - cfg.sweep_max
    if cfg.recipe == "cfg1":
        return [(2.0, 1000, 4, 3.0)]
    if cfg.recipe in ("cfg2", "cfg4"):
        out = []
        for _ in range(10):
            dm = float(g.uniform(5.0, 60.0))
            w = int(g.choice([1, 2, 4, 8]))
            a = float(g.uniform(0.5, 3.0))
            t0 = int(g.integers(0, nso - w))
            out.append((dm, t0, w, a))
        return out
    if cfg.recipe == "cfg5":
        out = []
        for _ in range(20):
            dm = float(g.uniform(5.0, 200.0))
            w = int(g.integers(1, 17))
            a = float(g.uniform(0.5, 3.0))
            t0 = int(g.integers(0, nso - w))
            out.append((dm, t0, w, a))
        return out
    raise ValueError(cfg.recipe)


def generate_beam(cfg: Config, b: int) -> np.ndarray:
    """One beam [nchans][nsamps] of cfg (float32 or uint8)."""
    seed = cfg.seed + b
    x = _noise(seed, cfg.nchans, cfg.nsamps)
    g = np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, 11])))
    if cfg.recipe == "cfg1":
        for (dm, t0, w, a) in pulses(cfg, b):
            _inject(x, cfg, dm, t0, w, a)
        return x
    if cfg.recipe == "cfg2":
        gain = g.uniform(0.5, 1.5, size=cfg.nchans).astype(np.float32)
        for (dm, t0, w, a) in pulses(cfg, b):
            _inject(x, cfg, dm, t0, w, a)
        x *= gain[:, None]
        return x
    if cfg.recipe == "cfg5":
        for (dm, t0, w, a) in pulses(cfg, b):
            _inject(x, cfg, dm, t0, w, a)
        return x
    if cfg.recipe == "cfg4":
        # noise quantised around mean 64, sigma 10; narrowband + broadband RFI; pulses x10
        x *= np.float32(10.0)
        x += np.float32(64.0)
        for (dm, t0, w, a) in pulses(cfg, b):
            _inject(x, cfg, dm, t0, w, 10.0 * a)
        t = np.arange(cfg.nsamps, dtype=np.float64)
        chans = g.choice(cfg.nchans, size=12, replace=False)
        for c in chans:
            P = g.uniform(2000.0, 20000.0)
            phi = g.uniform(0.0, 2 * np.pi)
            x[c] += (40.0 + 15.0 * np.sin(2 * np.pi * t / P + phi)).astype(np.float32)
        for _ in range(50):
            ts = int(g.integers(0, cfg.nsamps - 3))
            dur = int(g.integers(1, 4))
            x[:, ts:ts + dur] += np.float32(80.0)
        np.rint(x, out=x)
        np.clip(x, 0.0, 255.0, out=x)
        return x.astype(np.uint8)
    raise ValueError(cfg.recipe)


def generate(cfg: Config, beams=None) -> np.ndarray:
    """All (or the listed) beams stacked: [nb][nchans][nsamps]."""
    beams = range(cfg.nbeams) if beams is None else beams
    out = np.empty((len(beams), cfg.nchans, cfg.nsamps), dtype=cfg.np_dtype)
    for i, b in enumerate(beams):
        out[i] = generate_beam(cfg, b)
    return out


def generate_beam_device(cfg: Config, b: int, torch):
    """One beam [nchans][nsamps] of cfg's recipe drawn ON THE DEVICE with a seeded torch.Generator (config 5
    is generated on-device).  Same shapes, value distributions and injected structure as generate_beam, but another
    random stream: bench.py times on it; parity tests use generate_beam, whose arrays reach the oracle too."""
    gen = torch.Generator(device="cuda").manual_seed(cfg.seed + b)
    x = torch.empty((cfg.nchans, cfg.nsamps), dtype=torch.float32, device="cuda")
    x.normal_(generator=gen)
    g = np.random.Generator(np.random.PCG64(np.random.SeedSequence([cfg.seed + b, 11])))
    chan = torch.arange(cfg.nchans, device="cuda")

    def inject(scale):
        for (dm, t0, w, a) in pulses(cfg, b):
            sw = torch.from_numpy(cfg.sweep(dm)).cuda()
            for i in range(w):
                t = t0 + sw + i
                ok = t < cfg.nsamps
                x[chan[ok], t[ok]] += scale * a

    if cfg.recipe in ("cfg1", "cfg5"):
        inject(1.0)
        return x
    if cfg.recipe == "cfg2":
        inject(1.0)
        gain = torch.from_numpy(g.uniform(0.5, 1.5, size=cfg.nchans).astype(np.float32)).cuda()
        x *= gain[:, None]
        return x
    if cfg.recipe == "cfg4":
        x.mul_(10.0).add_(64.0)
        inject(10.0)
        t = torch.arange(cfg.nsamps, dtype=torch.float64, device="cuda")
        for c in g.choice(cfg.nchans, size=12, replace=False):
            P = g.uniform(2000.0, 20000.0)
            phi = g.uniform(0.0, 2 * np.pi)
            x[int(c)] += (40.0 + 15.0 * torch.sin(2 * np.pi * t / P + phi)).float()
        for _ in range(50):
            ts = int(g.integers(0, cfg.nsamps - 3))
            dur = int(g.integers(1, 4))
            x[:, ts:ts + dur] += 80.0
        return x.round_().clamp_(0.0, 255.0).to(torch.uint8)
    raise ValueError(cfg.recipe)


def power_filterbank(nbeams: int, nchans: int, nsamps: int, seed: int, window: int = 64) -> np.ndarray:
    """Detected-power filterbank for the paper's bandpass-fit RFI stage: exponentially distributed
    power (one detected sample of a Gaussian voltage) scaled by a smooth telescope bandpass with a small ripple, a few
    persistent narrow-band RFI channels (the ones the fit must mask), bursts of narrow-band RFI confined to single
    chunks of `window` samples and a few broadband spikes.  Inputs only: no pipeline arithmetic."""
    x = np.empty((nbeams, nchans, nsamps), dtype=np.float32)
    u = np.linspace(-1.0, 1.0, nchans)
    for b in range(nbeams):
        g = np.random.default_rng(seed + b)
        bp = 10.0 * (1.0 - 0.35 * u * u + 0.1 * u + 0.05 * u ** 3) * (1.0 + 0.01 * np.sin(40.0 * u + g.uniform(0, 6.28)))
        xb = g.exponential(size=(nchans, nsamps)).astype(np.float32) * bp[:, None].astype(np.float32)
        for c in g.choice(nchans, size=max(1, nchans // 100), replace=False):
            xb[c] *= np.float32(g.uniform(3.0, 8.0))                        # persistent RFI channels
        nchunk = nsamps // window
        for _ in range(max(2, nchans // 20)):
            c, j = int(g.integers(nchans)), int(g.integers(nchunk))
            xb[c, j * window:(j + 1) * window] += np.float32(bp[c] * g.uniform(1.0, 4.0))   # bursts
        for _ in range(5):
            xb[:, int(g.integers(nsamps))] += (bp * g.uniform(3.0, 6.0)).astype(np.float32)  # broadband spikes
        x[b] = xb
    return x
