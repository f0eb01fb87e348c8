"""Seeded synthetic frame-stack generator (inputs only; holds none of the QLD arithmetic).

The paper's camera recordings and its simulation (frame size, source
size and sampling interval unstated) are not available, so synthetic stacks with the paper's sensor
format (16-bit intensity frames), frame-size range and scene types stand in for them:
modulated point sources among unmodulated clutter, a scene under modulated
illumination and a translating object, as restated by
BASELINE.json `configs[0..4]`.  DESIGN.md section "Input recipe" lists every choice made here.

This module serves the tests, the oracle side and the CUDA side alike.  It is pure numpy.  A
sample x(s, p) of frame s (1-based) and pixel p (row-major index) is a pure function
of (scene, s, p), so any frame, any pixel's time series, or any subset can be produced
independently and in any order.  The per-sample recipe uses only integer hashing and IEEE-754
correctly-rounded double operations (+, *, sqrt, round-half-even), one rounding per operation, so
the device-side filler in csrc/synth_fill.cu reproduces it bit for bit:

    c      = (s * HW + p)                                  (uint64 counter)
    h_a    = mix64(key + (2c)   * GOLDEN)                  (splitmix64 stream)
    h_b    = mix64(key + (2c+1) * GOLDEN)
    t      = sum of the eight 16-bit fields of h_a, h_b    (integer, 0 .. 8*65535)
    z      = (t - 262140) * Z_SCALE                        (mean 0, variance 1, |z| < 4.9)
    lam    = base[p];  for j: lam = lam + weight_j[p] * mod_j[s]     (mul, then add)
             [+ disk_amp * mod_disk[s] if p lies inside the translating disk at frame s]
    x      = clamp(rint(lam + sqrt(noise_a + noise_b * lam) * z), 0, maxval)

noise_b = 1, noise_a = 0 is the rounded normal approximation N(lam, lam) of Poisson noise (all
means here are >= 100); noise_b = 0 is Gaussian noise of fixed variance noise_a.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Sequence, Tuple

import numpy as np

GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
# 1 / sqrt(8 * (65536^2 - 1) / 12): standard deviation of the sum of eight uniform 16-bit fields
Z_SCALE = 1.8688123650118534e-05
Z_OFFSET = 262140  # 8 * 65535 / 2


def mix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on uint64 arrays (wrapping arithmetic)."""
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = (x ^ (x >> np.uint64(30))) * _M1
        x = (x ^ (x >> np.uint64(27))) * _M2
        x = x ^ (x >> np.uint64(31))
    return x


def seed_key(seed: int, stream: int = 1) -> np.uint64:
    """Key of a noise stream; stream 0 draws the scene, stream 1 the per-sample noise."""
    with np.errstate(over="ignore"):
        k = mix64(np.uint64(seed) * GOLDEN + np.uint64(stream))
        return np.uint64(mix64(k + GOLDEN))


def _field_sum(h: np.ndarray) -> np.ndarray:
    m = np.uint64(0xFFFF)
    return ((h & m) + ((h >> np.uint64(16)) & m) + ((h >> np.uint64(32)) & m) + (h >> np.uint64(48))).astype(np.int64)


def unit_normal(key: np.uint64, counter: np.ndarray) -> np.ndarray:
    """z(counter): approximately N(0,1), exactly reproducible (see module docstring)."""
    c = np.asarray(counter, dtype=np.uint64)
    with np.errstate(over="ignore"):
        ha = mix64(key + (c * np.uint64(2)) * GOLDEN)
        hb = mix64(key + (c * np.uint64(2) + np.uint64(1)) * GOLDEN)
    t = _field_sum(ha) + _field_sum(hb)
    return (t - Z_OFFSET).astype(np.float64) * Z_SCALE


def unit_uniform(key: np.uint64, counter: np.ndarray) -> np.ndarray:
    """u(counter) in [0, 1) with 53 bits; used only for scene parameters (stream 0)."""
    c = np.asarray(counter, dtype=np.uint64)
    with np.errstate(over="ignore"):
        h = mix64(key + c * GOLDEN)
    return (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


@dataclass
class Disk:
    """Translating disk (PAPER.md:79-85 moving object): centre column (x0 + s) mod W, row cy."""
    x0: int
    cy: int
    radius: int
    amp: float            # counts
    mod: np.ndarray       # float64 [n_frames + 1], indexed by s


@dataclass
class Scene:
    H: int
    W: int
    n_frames: int                       # frames s = 1 .. n_frames exist
    dtype: str                          # "u8" or "u16"
    maxval: int
    seed: int
    base: np.ndarray                    # float32 [H*W]
    weights: np.ndarray                 # float32 [J, H*W]
    mods: np.ndarray                    # float64 [J, n_frames + 1], indexed by s (entry 0 unused)
    noise_a: float = 0.0
    noise_b: float = 1.0
    disk: Optional[Disk] = None
    meta: dict = field(default_factory=dict)

    @property
    def HW(self) -> int:
        return self.H * self.W

    @property
    def np_dtype(self):
        return np.uint8 if self.dtype == "u8" else np.uint16

    @property
    def key(self) -> np.uint64:
        return seed_key(self.seed, 1)


def _samples(scene: Scene, s: np.ndarray, p: np.ndarray) -> np.ndarray:
    """x(s, p) for broadcastable integer arrays s (1-based frame) and p (pixel index)."""
    s = np.asarray(s, dtype=np.int64)
    p = np.asarray(p, dtype=np.int64)
    s_b, p_b = np.broadcast_arrays(s, p)
    counter = (s_b.astype(np.uint64) * np.uint64(scene.HW) + p_b.astype(np.uint64))
    z = unit_normal(scene.key, counter)
    lam = scene.base.astype(np.float64)[p_b]
    for j in range(scene.weights.shape[0]):
        lam = lam + scene.weights[j].astype(np.float64)[p_b] * scene.mods[j][s_b]
    if scene.disk is not None:
        d = scene.disk
        px = p_b % scene.W
        py = p_b // scene.W
        dx = (px - d.x0 - s_b) % scene.W          # python-style non-negative modulo
        dx = np.where(dx >= scene.W - dx, dx - scene.W, dx)   # wrap to [-W/2, W/2)
        dy = py - d.cy
        inside = (dx * dx + dy * dy) <= d.radius * d.radius
        lam = np.where(inside, lam + d.amp * d.mod[s_b], lam)
    var = scene.noise_a + scene.noise_b * lam
    x = np.rint(lam + np.sqrt(var) * z)
    x = np.clip(x, 0.0, float(scene.maxval))
    return x.astype(scene.np_dtype)


def frames(scene: Scene, s_first: int, n: int) -> np.ndarray:
    """Frames s_first .. s_first+n-1 as an array [n, H, W] of the scene's dtype."""
    assert 1 <= s_first and s_first + n - 1 <= scene.n_frames
    out = np.empty((n, scene.HW), dtype=scene.np_dtype)
    p = np.arange(scene.HW, dtype=np.int64)
    for i in range(n):
        out[i] = _samples(scene, np.int64(s_first + i), p)
    return out.reshape(n, scene.H, scene.W)


def series(scene: Scene, pixels: Sequence[int], s_first: int = 1, n: Optional[int] = None) -> np.ndarray:
    """Time series of the given pixel indices: array [n, len(pixels)]."""
    if n is None:
        n = scene.n_frames - s_first + 1
    s = np.arange(s_first, s_first + n, dtype=np.int64)[:, None]
    p = np.asarray(pixels, dtype=np.int64)[None, :]
    return _samples(scene, s, p)


# ----------------------------------------------------------------------------------------------
# scene construction helpers (stream 0 of the seed)
# ----------------------------------------------------------------------------------------------
class _SceneRng:
    def __init__(self, seed: int):
        self.key = seed_key(seed, 0)
        self.n = 0

    def uniform(self, lo: float = 0.0, hi: float = 1.0) -> float:
        u = float(unit_uniform(self.key, np.uint64(self.n)))
        self.n += 1
        return lo + (hi - lo) * u

    def normal_field(self, size: int) -> np.ndarray:
        c = np.arange(self.n, self.n + size, dtype=np.uint64)
        self.n += size
        return unit_normal(self.key, c)


def _gauss_spot(H: int, W: int, cx: float, cy: float, sigma: float) -> np.ndarray:
    y = np.arange(H, dtype=np.float64)[:, None]
    x = np.arange(W, dtype=np.float64)[None, :]
    return np.exp(-((x - cx) ** 2 + (y - cy) ** 2) / (2.0 * sigma * sigma))


def _place_points(rng: _SceneRng, H: int, W: int, count: int, margin: float, min_sep: float,
                  taken: list) -> list:
    """Uniform positions at least `margin` from the edges and `min_sep` from each other."""
    pts = []
    margin = min(margin, 0.25 * min(H, W))
    guard = 0
    while len(pts) < count:
        cx = rng.uniform(margin, W - 1 - margin)
        cy = rng.uniform(margin, H - 1 - margin)
        guard += 1
        ok = all((cx - a) ** 2 + (cy - b) ** 2 >= min_sep ** 2 for a, b in taken + pts)
        if ok or guard > 1000:
            pts.append((cx, cy))
    return pts


def _tone(nu_num: float, nu_den: float, n_frames: int, phase: float) -> np.ndarray:
    s = np.arange(n_frames + 1, dtype=np.float64)
    return np.sin(2.0 * np.pi * (nu_num * s / nu_den) + phase)


@dataclass
class Workload:
    """A scene plus the demodulation parameters BASELINE.json names for it."""
    name: str
    scene: Scene
    N: int                                    # window length
    refs: Tuple[dict, ...]                    # each: {"nu": float, "num": int, "den": int, "phase": float}
    hop: int = 0                              # > 0: sliding window
    batch: int = 0                            # frames per push (streaming)


def cfg0(H: int = 64, W: int = 64, N: int = 64, seed: int = 0) -> Workload:
    """BASELINE.json configs[0]: u8, nu = 1/4, background 100 + N(0, 5^2), radius-12 disk, 2 counts."""
    base = np.full(H * W, 100.0, dtype=np.float32)
    y, x = np.mgrid[0:H, 0:W]
    r = 12.0 * min(H, W) / 64.0
    disk = ((x - W // 2) ** 2 + (y - H // 2) ** 2 <= r * r).astype(np.float32).reshape(-1)
    mods = _tone(1.0, 4.0, N, 0.0)[None, :]
    sc = Scene(H, W, N, "u8", 255, seed, base, (2.0 * disk)[None, :].astype(np.float32), mods,
               noise_a=25.0, noise_b=0.0, meta={"disk_mask": disk.astype(bool)})
    return Workload("cfg0", sc, N, ({"nu": 0.25, "num": 1, "den": 4, "phase": 0.0},))


def cfg1(H: int = 480, W: int = 640, N: int = 256, seed: int = 1) -> Workload:
    """configs[1]: u8, nu = 1/8, Poisson(120), 5 modulated spots (0.5 counts), 3 clutter spots (peak 200)."""
    rng = _SceneRng(seed)
    sigma = 3.0
    src = _place_points(rng, H, W, 5, 4 * sigma, 8 * sigma, [])
    clu = _place_points(rng, H, W, 3, 4 * sigma, 8 * sigma, src)
    base = np.full((H, W), 120.0)
    for cx, cy in clu:
        base += 80.0 * _gauss_spot(H, W, cx, cy, sigma)
    weights = np.stack([0.5 * _gauss_spot(H, W, cx, cy, sigma).reshape(-1) for cx, cy in src])
    phases = [rng.uniform(0.0, 2.0 * np.pi) for _ in src]
    mods = np.stack([_tone(1.0, 8.0, N, ph) for ph in phases])
    sc = Scene(H, W, N, "u8", 255, seed, base.reshape(-1).astype(np.float32), weights.astype(np.float32), mods,
               meta={"sources": src, "clutter": clu, "phases": phases})
    return Workload("cfg1", sc, N, ({"nu": 0.125, "num": 1, "den": 8, "phase": 0.0},))


def _smooth_field(rng: _SceneRng, H: int, W: int, sigma: float) -> np.ndarray:
    from scipy.ndimage import gaussian_filter
    white = rng.normal_field(H * W).reshape(H, W)
    f = gaussian_filter(white, sigma=min(sigma, 0.25 * min(H, W)), mode="wrap")
    f = (f - f.mean()) / f.std()
    return f


def cfg2(H: int = 1024, W: int = 1280, N: int = 1024, seed: int = 2, nu: float = 0.0937) -> Workload:
    """configs[2]: u16 (12-bit), nu = 0.0937, smooth background (mean 2000), Poisson, 20 % mask at 5 counts."""
    rng = _SceneRng(seed)
    base = 2000.0 + 200.0 * _smooth_field(rng, H, W, 50.0)
    mask = np.zeros((H, W), dtype=bool)
    lo, hi = max(2, 16 * min(H, W) // 1024), max(4, 128 * min(H, W) // 1024)
    guard = 0
    while mask.mean() < 0.195 and guard < 100000:
        h = int(rng.uniform(lo, hi + 1)); w = int(rng.uniform(lo, hi + 1))
        y0 = int(rng.uniform(0, max(1, H - h))); x0 = int(rng.uniform(0, max(1, W - w)))
        mask[y0:y0 + h, x0:x0 + w] = True
        guard += 1
    phase = rng.uniform(0.0, 2.0 * np.pi)
    s = np.arange(N + 1, dtype=np.float64)
    mods = np.sin(2.0 * np.pi * nu * s + phase)[None, :]
    weights = (5.0 * mask.reshape(-1))[None, :].astype(np.float32)
    sc = Scene(H, W, N, "u16", 4095, seed, base.reshape(-1).astype(np.float32), weights, mods,
               meta={"mask": mask, "phase": phase})
    return Workload("cfg2", sc, N, ({"nu": nu, "num": 0, "den": 0, "phase": 0.0},))


def cfg3(H: int = 1024, W: int = 1024, n_stream: int = 16384, N: int = 512, hop: int = 32, batch: int = 32,
         seed: int = 3) -> Workload:
    """configs[3]: u16 (12-bit) stream, nu = 1/6, Poisson(1500), radius-40 disk at 3 counts moving 1 px/frame."""
    rng = _SceneRng(seed)
    phase = rng.uniform(0.0, 2.0 * np.pi)
    x0 = int(rng.uniform(0, W))
    base = np.full(H * W, 1500.0, dtype=np.float32)
    radius = max(2, 40 * min(H, W) // 1024)
    disk = Disk(x0=x0, cy=H // 2, radius=radius, amp=3.0, mod=_tone(1.0, 6.0, n_stream, phase))
    sc = Scene(H, W, n_stream, "u16", 4095, seed, base, np.zeros((0, H * W), np.float32),
               np.zeros((0, n_stream + 1)), disk=disk, meta={"phase": phase, "x0": x0})
    return Workload("cfg3", sc, N, ({"nu": 1.0 / 6.0, "num": 1, "den": 6, "phase": 0.0},), hop=hop, batch=batch)


def cfg4(H: int = 2048, W: int = 2048, N: int = 2048, K: int = 8, seed: int = 4) -> Workload:
    """configs[4]: u16 (12-bit), K = 8 spots at distinct nu in [0.05, 0.45], 20 clutter spots, Poisson(1000)."""
    rng = _SceneRng(seed)
    sigma = max(1.0, 6.0 * min(H, W) / 2048.0)
    src = _place_points(rng, H, W, K, 4 * sigma, 8 * sigma, [])
    clu = _place_points(rng, H, W, 20, 4 * sigma, 8 * sigma, src)
    base = np.full((H, W), 1000.0)
    for cx, cy in clu:
        base += 500.0 * _gauss_spot(H, W, cx, cy, sigma)
    nus = [0.05 + 0.4 * (k + rng.uniform(0.1, 0.9)) / K for k in range(K)]
    phases = [rng.uniform(0.0, 2.0 * np.pi) for _ in range(K)]
    amps = [rng.uniform(1.0, 4.0) for _ in range(K)]
    weights = np.stack([amps[k] * _gauss_spot(H, W, src[k][0], src[k][1], sigma).reshape(-1) for k in range(K)])
    s = np.arange(N + 1, dtype=np.float64)
    mods = np.stack([np.sin(2.0 * np.pi * nus[k] * s + phases[k]) for k in range(K)])
    sc = Scene(H, W, N, "u16", 4095, seed, base.reshape(-1).astype(np.float32), weights.astype(np.float32), mods,
               meta={"sources": src, "clutter": clu, "nus": nus, "phases": phases, "amps": amps})
    refs = tuple({"nu": float(nus[k]), "num": 0, "den": 0, "phase": 0.0} for k in range(K))
    return Workload("cfg4", sc, N, refs)


BUILDERS = {"cfg0": cfg0, "cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg4": cfg4}


# ----------------------------------------------------------------------------------------------
# The paper's own numerical simulation (Fig. 1): SURVEY.md 8(f1), a second workload
# ----------------------------------------------------------------------------------------------
@dataclass
class PaperSim:
    """Frames of the five-source scene plus where the sources sit."""
    frames: np.ndarray                        # [N, n, n] uint16
    boxes: Tuple[Tuple[int, int], ...]        # top-left (y0, x0) of the five m x m sub-regions; the last one is constant
    m: int
    nus: Tuple[float, ...]                    # f_i / f_s of the four modulated sources
    gain: float
    X: float


def paper_sim(n: int = 96, m: int = 8, N: int = 82, X: float = 5.0, nus: Sequence[float] = (0.20, 0.23, 0.26, 0.29),
              seed: int = 7, gain: float = 1000.0) -> PaperSim:
    """an n x n frame with five non-overlapping m x m sub-regions; in four of them the intensity is
    (0.5 + sin(omega_i t_s)), t_s = s dt, s = 1..N, the fifth is held constant; every pixel of every frame gets an
    independent random number uniform in [0, X] (X in 1..10 in the paper).
    The paper does not give n, m, dt or the noise generator; the defaults here are this build's choice (DESIGN.md
    reading G21): frequencies 20/23/26/29 Hz at an assumed 100 frames/s, N = 82
    (PAPER.md:37).  Intensities are real numbers in the paper; the device path takes integers, so the frame is
    x = rint(gain * (intensity + 0.5)) as uint16 -- an affine map, which leaves Eq. (1)'s CNR of a map that is linear
    in the data unchanged and only adds the constant-background leakage of reading G9."""
    assert n >= 9 * m and len(nus) == 4
    # five boxes: four around the centre of each quadrant's inner half and one in the middle, each with room for
    # the m-wide surround of Fig. 6
    c = [(n // 4, n // 4), (n // 4, 3 * n // 4), (3 * n // 4, n // 4), (3 * n // 4, 3 * n // 4), (n // 2, n // 2)]
    boxes = tuple((cy - m // 2, cx - m // 2) for cy, cx in c)
    key = seed_key(seed, 1)
    s = np.arange(1, N + 1, dtype=np.int64)[:, None]
    p = np.arange(n * n, dtype=np.int64)[None, :]
    u = unit_uniform(key, (s.astype(np.uint64) * np.uint64(n * n) + p.astype(np.uint64)))
    inten = (X * u).reshape(N, n, n)
    t = np.arange(1, N + 1, dtype=np.float64)
    for i, (y0, x0) in enumerate(boxes):
        src = (0.5 + np.sin(2.0 * np.pi * nus[i] * t)) if i < 4 else np.full(N, 1.5)
        inten[:, y0:y0 + m, x0:x0 + m] += src[:, None, None]
    x = np.clip(np.rint(gain * (inten + 0.5)), 0, 65535).astype(np.uint16)
    return PaperSim(x, boxes, m, tuple(float(v) for v in nus), float(gain), float(X))
