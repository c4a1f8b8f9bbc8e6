"""Seeded synthetic radio-sky image pairs -- the ONLY module shared by the CUDA path's
harness and the oracle's tests.  It holds none of the method's arithmetic (no clamp, no
LISI/augLISI term, no reduction): it only draws inputs.

The paper evaluates on OSKAR-simulated, CLEAN-restored SKA1-LOW images of GLEAM sources
(Sec. 3: 2048 x 2048 pixels, 33 sources in MS1, 5 low-intensity sources
removed in MS2; tiles of 64 x 64).  None of that data is available, so
these seeded skies stand in for it, with the shapes and statistics BASELINE.json's five
configs prescribe.  The recipe (also in DESIGN.md, "Input recipe"):

  image  = sum of sources + zero-mean Gaussian noise  (about half the pixels are negative
           before the clamp, away from sources)
  point source    amp * exp(-((r-cy)^2 + (c-cx)^2) / (2 sigma^2)), window +-ceil(6 sigma)
  extended source amp * exp(-(u^2/sa^2 + v^2/sb^2)/2), (u,v) rotated by theta~U[0,pi),
                  sa, sb ~ U(5,40) px, amp log-uniform 1e-3..1e-1, window +-ceil(5 max(sa,sb))
  positions       (cy, cx) ~ U[0,N)^2 ; pixel (r,c) has centre (r,c)
  flux laws       log-uniform: amp = 10^U(log10 lo, log10 hi)
                  power law index -1.8 on [lo,hi] by inverse CDF
  pair            base = the sources common to x and y, rendered once in fp32 (each patch
                  evaluated in fp64); x = base + changed sources at their x amplitude +
                  noise_x ; y = base + changed sources at their y amplitude (0 when the
                  source is removed, factor*amp when it varies) + noise_y, with independent
                  noise realisations ("fresh noise").
  RNG             numpy Philox keyed by (seed, stream id): positions / fluxes / extended
                  parameters / selection / noise-x / noise-y are separate streams, so the
                  image does not depend on N_T.  With ``device="cuda"`` the noise is drawn by
                  a seeded torch CUDA generator instead (same recipe, different realisation;
                  the finished buffers are the source of truth for both sides).
  time series     ``make_series``: M snapshots of one field ("on-and-off emission
                  behaviour ... between observations of the same section of the sky").  The sources
                  the config's change rule selects are the transients; snapshot 0 shows all of them
                  in their x state (MS1), and in every later snapshot each transient is, with
                  probability 1/2, in its y state (absent / scaled) instead; fixed sources never
                  change; every snapshot has fresh noise.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np

_STREAMS = {"pos": 1, "flux": 2, "ext": 3, "select": 4, "noise_x": 5, "noise_y": 6, "series": 7}
_NOISE_SNAPSHOT0 = 100         # snapshot j of a series draws its noise from stream 100 + j


def _rng(seed: int, stream) -> np.random.Generator:
    sid = _STREAMS[stream] if isinstance(stream, str) else int(stream)
    return np.random.Generator(np.random.Philox(key=[int(seed), sid]))


@dataclass(frozen=True)
class SkyConfig:
    name: str
    N: int
    N_T: int
    n_point: int
    psf_sigma: float
    flux_law: str                  # "loguniform" | "powerlaw"
    flux_lo: float
    flux_hi: float
    noise_sigma: float
    n_ext: int = 0
    change: str = "drop_faintest"  # "drop_faintest" | "drop_and_scale" | "drop_fraction"
    n_drop: int = 5
    n_scale: int = 0
    drop_fraction: float = 0.0
    seed: int = 0
    C1: float = 1e-6
    C2: float = 1e-6
    C: float = 1e-6
    n_pairs: int = 1               # config [4]: throughput loop over 16 pairs (seeds 0..15)
    sweep_N_T: tuple = field(default_factory=tuple)

    @property
    def D(self) -> float:
        # Reading R1: D = C1/2 makes LISI(x, x) -> 1.
        return float(np.float32(self.C1)) / 2.0


# BASELINE.json "configs", index by index.
CONFIGS = {
    0: SkyConfig("cfg0_N256_T16", 256, 16, 30, 1.5, "loguniform", 1e-3, 1.0, 1e-4, seed=0),
    1: SkyConfig("cfg1_N2048_T64", 2048, 64, 33, 2.0, "powerlaw", 1e-3, 2.0, 1e-4, seed=0),
    2: SkyConfig("cfg2_N2048_sweep", 2048, 64, 33, 2.0, "powerlaw", 1e-3, 2.0, 1e-4, seed=1,
                 sweep_N_T=(8, 16, 32, 64, 128, 256, 512)),
    3: SkyConfig("cfg3_N8192_T64", 8192, 64, 2000, 2.0, "powerlaw", 1e-3, 2.0, 1e-3, n_ext=50,
                 change="drop_and_scale", n_drop=20, n_scale=20, seed=0),
    4: SkyConfig("cfg4_N16384_T128", 16384, 128, 20000, 2.0, "powerlaw", 1e-3, 2.0, 1e-3,
                 n_ext=500, change="drop_fraction", drop_fraction=0.01, seed=0, n_pairs=16),
}


def scaled(cfg: SkyConfig, N: int, N_T: int | None = None) -> SkyConfig:
    """The same recipe on a smaller canvas (source counts scaled with the area) -- used by
    CPU-only tests that need a config-[3]/[4]-like sky the oracle finishes in seconds."""
    f = (N / cfg.N) ** 2
    return replace(cfg, name=f"{cfg.name}_scaled{N}", N=N, N_T=N_T or cfg.N_T,
                   n_point=max(8, int(round(cfg.n_point * f))),
                   n_ext=int(round(cfg.n_ext * f)),
                   n_drop=min(cfg.n_drop, max(1, int(round(cfg.n_point * f)) // 4)),
                   n_scale=min(cfg.n_scale, max(0, int(round(cfg.n_point * f)) // 4)))


def _draw_sources(cfg: SkyConfig, seed: int) -> dict:
    N = cfg.N
    rp, rf, re = _rng(seed, "pos"), _rng(seed, "flux"), _rng(seed, "ext")
    n = cfg.n_point + cfg.n_ext
    cy = rp.uniform(0.0, N, n)
    cx = rp.uniform(0.0, N, n)
    u = rf.uniform(0.0, 1.0, cfg.n_point)
    if cfg.flux_law == "loguniform":
        amp_p = 10.0 ** (math.log10(cfg.flux_lo) + u * (math.log10(cfg.flux_hi) - math.log10(cfg.flux_lo)))
    elif cfg.flux_law == "powerlaw":      # dN/df ~ f^-1.8  ->  CDF in f^-0.8
        a, b = cfg.flux_lo ** -0.8, cfg.flux_hi ** -0.8
        amp_p = (a + u * (b - a)) ** (-1.0 / 0.8)
    else:
        raise ValueError(cfg.flux_law)
    sa = np.full(n, cfg.psf_sigma)
    sb = np.full(n, cfg.psf_sigma)
    th = np.zeros(n)
    amp = np.empty(n)
    amp[:cfg.n_point] = amp_p
    if cfg.n_ext:
        sa[cfg.n_point:] = re.uniform(5.0, 40.0, cfg.n_ext)
        sb[cfg.n_point:] = re.uniform(5.0, 40.0, cfg.n_ext)
        th[cfg.n_point:] = re.uniform(0.0, math.pi, cfg.n_ext)
        amp[cfg.n_point:] = 10.0 ** re.uniform(-3.0, -1.0, cfg.n_ext)
    return {"cy": cy, "cx": cx, "amp": amp, "sa": sa, "sb": sb, "theta": th,
            "is_ext": np.arange(n) >= cfg.n_point}


def _select_changes(cfg: SkyConfig, src: dict, seed: int):
    """Return (amp_x, amp_y): per-source amplitudes in x and in y (0 = absent)."""
    rs = _rng(seed, "select")
    amp_x = src["amp"].copy()
    amp_y = src["amp"].copy()
    n = amp_x.size
    if cfg.change == "drop_faintest":            # configs 0-2: the n_drop lowest-flux sources vanish in y
        order = np.argsort(src["amp"][:cfg.n_point], kind="stable")
        amp_y[order[:cfg.n_drop]] = 0.0
    elif cfg.change == "drop_and_scale":         # config 3: 20 random point sources vanish, 20 others vary
        perm = rs.permutation(cfg.n_point)
        amp_y[perm[:cfg.n_drop]] = 0.0
        sel = perm[cfg.n_drop:cfg.n_drop + cfg.n_scale]
        amp_y[sel] = amp_x[sel] * rs.uniform(0.5, 1.5, sel.size)
    elif cfg.change == "drop_fraction":          # config 4: 1 % of all sources vanish
        k = int(round(cfg.drop_fraction * n))
        amp_y[rs.permutation(n)[:k]] = 0.0
    else:
        raise ValueError(cfg.change)
    return amp_x, amp_y


def _render(img: np.ndarray, src: dict, amps: np.ndarray, idx) -> None:
    """Add the sources ``idx`` with amplitudes ``amps[idx]`` into the fp32 image, patch by patch."""
    N = img.shape[0]
    for i in idx:
        a = float(amps[i])
        if a == 0.0:
            continue
        cy, cx = float(src["cy"][i]), float(src["cx"][i])
        sa, sb, th = float(src["sa"][i]), float(src["sb"][i]), float(src["theta"][i])
        half = math.ceil((5.0 if src["is_ext"][i] else 6.0) * max(sa, sb))
        r0, r1 = max(0, int(math.floor(cy)) - half), min(N, int(math.floor(cy)) + half + 1)
        c0, c1 = max(0, int(math.floor(cx)) - half), min(N, int(math.floor(cx)) + half + 1)
        if r0 >= r1 or c0 >= c1:
            continue
        dy = (np.arange(r0, r1, dtype=np.float64) - cy)[:, None]
        dx = (np.arange(c0, c1, dtype=np.float64) - cx)[None, :]
        ct, st = math.cos(th), math.sin(th)
        u = ct * dx + st * dy
        v = -st * dx + ct * dy
        img[r0:r1, c0:c1] += a * np.exp(-0.5 * (u * u / (sa * sa) + v * v / (sb * sb)))


def sky_layers(cfg: SkyConfig, seed: int | None = None):
    """Noise-free fp32 layers (x_sky, y_sky) and the source table (with amp_x / amp_y)."""
    seed = cfg.seed if seed is None else seed
    src = _draw_sources(cfg, seed)
    amp_x, amp_y = _select_changes(cfg, src, seed)
    same = amp_x == amp_y
    base = np.zeros((cfg.N, cfg.N), dtype=np.float32)
    _render(base, src, amp_x, np.nonzero(same)[0])
    x = base.copy()
    y = base
    changed = np.nonzero(~same)[0]
    _render(x, src, amp_x, changed)
    _render(y, src, amp_y, changed)
    src = dict(src, amp_x=amp_x, amp_y=amp_y)
    return x, y, src


def _add_noise_host(img: np.ndarray, sigma: float, rng: np.random.Generator) -> None:
    rows = max(1, (1 << 24) // img.shape[1])
    for r in range(0, img.shape[0], rows):
        blk = img[r:r + rows]
        blk += np.float32(sigma) * rng.standard_normal(blk.shape, dtype=np.float32)


def make_pair(cfg: SkyConfig, seed: int | None = None, device: str | None = None,
              shared_noise: bool = False):
    """Build one image pair.  Host (default): two C-contiguous float32 numpy arrays.
    ``device="cuda"``: two torch CUDA tensors (sky rendered on the host and uploaded, noise
    drawn on the device).  ``shared_noise=True`` gives y the SAME noise as x (the
    "shared-noise" parity variant: x == y exactly away from the changed sources, so
    |x-y| = 0 there and the Eq. 1 terms reach (x+y)/C1).
    Returns (x, y, meta)."""
    seed = cfg.seed if seed is None else seed
    x, y, src = sky_layers(cfg, seed)
    meta = {"cfg": cfg, "seed": seed, "sources": src}
    if device is None:
        if shared_noise:
            noise = np.zeros_like(x)
            _add_noise_host(noise, cfg.noise_sigma, _rng(seed, "noise_x"))
            x += noise
            y += noise
        else:
            _add_noise_host(x, cfg.noise_sigma, _rng(seed, "noise_x"))
            _add_noise_host(y, cfg.noise_sigma, _rng(seed, "noise_y"))
        return x, y, meta
    import torch
    dev = torch.device(device)
    gx = torch.Generator(device=dev).manual_seed(2 * seed + 1)
    xt = torch.from_numpy(x).to(dev)
    yt = torch.from_numpy(y).to(dev)
    nx = torch.randn(xt.shape, generator=gx, device=dev, dtype=torch.float32)
    xt.add_(nx, alpha=cfg.noise_sigma)
    if shared_noise:
        yt.add_(nx, alpha=cfg.noise_sigma)
    else:
        del nx
        gy = torch.Generator(device=dev).manual_seed(2 * seed + 2)
        yt.add_(torch.randn(yt.shape, generator=gy, device=dev, dtype=torch.float32),
                alpha=cfg.noise_sigma)
    return xt, yt, meta


def make_series(cfg: SkyConfig, n_images: int, seed: int | None = None, device: str | None = None):
    """A time series of ``n_images`` snapshots of the config's sky (recipe in the module docstring).
    Host (default): list of C-contiguous float32 numpy arrays; ``device="cuda"``: list of torch CUDA
    tensors (sky rendered on the host, noise drawn on the device).  Returns (images, meta);
    ``meta["state_y"][j, i]`` tells whether changed source i is in its y state in snapshot j."""
    if n_images < 2:
        raise ValueError("a series needs at least two images")
    seed = cfg.seed if seed is None else seed
    src = _draw_sources(cfg, seed)
    amp_x, amp_y = _select_changes(cfg, src, seed)
    same = amp_x == amp_y
    changed = np.nonzero(~same)[0]
    base = np.zeros((cfg.N, cfg.N), dtype=np.float32)
    _render(base, src, amp_x, np.nonzero(same)[0])
    state_y = _rng(seed, "series").random((n_images, changed.size)) < 0.5
    state_y[0] = False                                  # snapshot 0: every transient in its x state
    images = []
    if device is not None:
        import torch
        dev = torch.device(device)
    for j in range(n_images):
        amps = amp_x.copy()
        amps[changed[state_y[j]]] = amp_y[changed[state_y[j]]]
        img = base.copy()
        _render(img, src, amps, changed)
        if device is None:
            _add_noise_host(img, cfg.noise_sigma, _rng(seed, _NOISE_SNAPSHOT0 + j))
            images.append(img)
        else:
            g = torch.Generator(device=dev).manual_seed(1000003 * seed + 17 * j + 5)
            t = torch.from_numpy(img).to(dev)
            t.add_(torch.randn(t.shape, generator=g, device=dev, dtype=torch.float32), alpha=cfg.noise_sigma)
            images.append(t)
    meta = {"cfg": cfg, "seed": seed, "sources": dict(src, amp_x=amp_x, amp_y=amp_y),
            "changed": changed, "state_y": state_y}
    return images, meta
