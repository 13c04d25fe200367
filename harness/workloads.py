"""Seeded synthetic workloads shaped like BASELINE.json's five configurations (C1..C5).

Input data only: occupancy bitmaps, robot specifications (footprint polygon, beam-angle table,
limits), task parameters, action tapes, reset seeds and forced-reset masks.  The recipes are the
ones in SURVEY.md section 8(d) ("Synthetic inputs") and are restated in DESIGN.md; they stand in for
the paper's maps SEnv1/SEnv2, which exist only as figures.

All generation is host-side NumPy with `default_rng(seed)`; resolution is 0.05 m/cell throughout.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

DRIVE_DIFF = 0
DRIVE_OMNI = 1
RHO = np.float32(0.05)


@dataclass
class Workload:
    name: str
    occ: np.ndarray                 # uint8 [H, W], !=0 occupied
    resolution: np.float32
    footprint: np.ndarray           # float32 [V, 2] body frame, metres, ordered
    beam_angles: np.ndarray         # float32 [B] rad, body frame
    max_range: np.float32
    drive: int
    vel_limits: np.ndarray          # float32 [6] vx_min,vx_max,vy_min,vy_max,w_min,w_max
    n_envs: int
    dt: np.float32
    steps: int
    seed: int
    goal_tol: np.float32 = np.float32(0.3)
    max_episode_steps: int = 0
    goal_dist_min: np.float32 = np.float32(3.0)
    goal_dist_max: np.float32 = np.float32(8.0)
    r_success: np.float32 = np.float32(10.0)
    r_collision: np.float32 = np.float32(-10.0)
    c_progress: np.float32 = np.float32(2.0)
    regions: np.ndarray | None = None   # int32 [n, 4] = row0, col0, h, w ; env e -> region e % n
    forced_reset_frac: float = 0.0
    ring_capacity: int = 0
    extra: dict = field(default_factory=dict)

    @property
    def action_dim(self) -> int:
        return 2 if self.drive == DRIVE_DIFF else 3

    @property
    def n_beams(self) -> int:
        return int(self.beam_angles.shape[0])


# ----------------------------------------------------------------------------- maps

def _border(occ: np.ndarray) -> None:
    occ[0, :] = 1
    occ[-1, :] = 1
    occ[:, 0] = 1
    occ[:, -1] = 1


def _add_rect(occ, rng, lo=2, hi=20) -> int:
    """Returns the number of newly occupied cells."""
    H, W = occ.shape
    h = int(rng.integers(lo, hi + 1))
    w = int(rng.integers(lo, hi + 1))
    r = int(rng.integers(0, H - h + 1))
    c = int(rng.integers(0, W - w + 1))
    new = h * w - int(occ[r:r + h, c:c + w].sum())
    occ[r:r + h, c:c + w] = 1
    return new


def _add_disc(occ, rng, rlo, rhi, window=None) -> int:
    H, W = occ.shape
    r0, c0, h, w = (0, 0, H, W) if window is None else window
    rad = float(rng.uniform(rlo, rhi))
    cy = float(rng.uniform(r0, r0 + h))
    cx = float(rng.uniform(c0, c0 + w))
    ra, rb = max(r0, int(cy - rad) - 1), min(r0 + h, int(cy + rad) + 2)
    ca, cb = max(c0, int(cx - rad) - 1), min(c0 + w, int(cx + rad) + 2)
    if ra >= rb or ca >= cb:
        return 0
    yy, xx = np.mgrid[ra:rb, ca:cb]
    m = (yy + 0.5 - cy) ** 2 + (xx + 0.5 - cx) ** 2 <= rad * rad
    sub = occ[ra:rb, ca:cb]
    new = int(m.sum()) - int(sub[m].sum())
    sub[m] = 1
    return new


def map_rectangles(size: int, frac: float, seed: int, n_discs: int = 0,
                   disc_r=(3.0, 10.0)) -> np.ndarray:
    """Border walls + axis-aligned rectangles (sides U{2..20}) until >= frac occupied, then discs."""
    rng = np.random.default_rng(seed)
    occ = np.zeros((size, size), np.uint8)
    _border(occ)
    filled, target = int(occ.sum()), frac * occ.size
    while filled < target:
        filled += _add_rect(occ, rng)
    for _ in range(n_discs):
        _add_disc(occ, rng, *disc_r)
    return occ


def map_large_maze(size: int, frac: float, seed: int) -> np.ndarray:
    """C4: rectangles and discs to `frac`, then one quadrant made solid and carved by a randomised
    depth-first maze whose corridors are U[20,40] cells (1-2 m) wide."""
    rng = np.random.default_rng(seed)
    occ = np.zeros((size, size), np.uint8)
    _border(occ)
    k = 0
    filled, target = int(occ.sum()), frac * occ.size
    while filled < target:
        if k % 4 == 3:
            filled += _add_disc(occ, rng, 3.0, 10.0)
        else:
            filled += _add_rect(occ, rng)
        k += 1
    q = size // 2
    pitch = 64
    g = q // pitch                      # maze cells per side
    r0, c0 = q, q                       # lower-right quadrant
    occ[r0:, c0:] = 1
    seen = np.zeros((g, g), bool)
    stack = [(0, 0)]
    seen[0, 0] = True

    def carve(ra, rb, ca, cb):
        ra, rb = max(ra, r0 + 1), min(rb, size - 1)
        ca, cb = max(ca, c0 + 1), min(cb, size - 1)
        occ[ra:rb, ca:cb] = 0

    def centre(i, j):
        return r0 + i * pitch + pitch // 2, c0 + j * pitch + pitch // 2

    w0 = int(rng.integers(20, 41))
    cy, cx = centre(0, 0)
    carve(cy - w0 // 2, cy + (w0 + 1) // 2, cx - w0 // 2, cx + (w0 + 1) // 2)
    while stack:
        i, j = stack[-1]
        nb = [(i + di, j + dj) for di, dj in ((1, 0), (-1, 0), (0, 1), (0, -1))
              if 0 <= i + di < g and 0 <= j + dj < g and not seen[i + di, j + dj]]
        if not nb:
            stack.pop()
            continue
        ni, nj = nb[int(rng.integers(0, len(nb)))]
        seen[ni, nj] = True
        w = int(rng.integers(20, 41))
        ay, ax = centre(i, j)
        by, bx = centre(ni, nj)
        lo, hi = w // 2, (w + 1) // 2
        carve(min(ay, by) - lo, max(ay, by) + hi, min(ax, bx) - lo, max(ax, bx) + hi)
        stack.append((ni, nj))
    # an opening from the maze's first cell into the open part of the map
    cy, cx = centre(0, 0)
    occ[cy - 15:cy + 15, c0 - 2:c0 + pitch // 2] = 0
    _border(occ)
    return occ


def map_tile_atlas(seed: int, n_tiles: int = 128, tile: int = 64, slots: int = 16):
    """C5: `slots` x `slots` atlas of `tile`^2-cell tiles; tiles 0..n_tiles-1 row-major, each with a
    1-cell border and random discs (radius U[2,6]) to a per-tile density U[10%,40%]; other slots solid."""
    rng = np.random.default_rng(seed)
    size = tile * slots
    occ = np.ones((size, size), np.uint8)
    regions = np.zeros((n_tiles, 4), np.int32)
    for t in range(n_tiles):
        r0, c0 = (t // slots) * tile, (t % slots) * tile
        sub = np.zeros((tile, tile), np.uint8)
        _border(sub)
        dens = float(rng.uniform(0.10, 0.40))
        filled = int(sub.sum())
        while filled < dens * sub.size:
            filled += _add_disc(sub, rng, 2.0, 6.0)
        _border(sub)
        occ[r0:r0 + tile, c0:c0 + tile] = sub
        regions[t] = (r0, c0, tile, tile)
    return occ, regions


# ----------------------------------------------------------------------------- robots

def footprint_ngon(radius: float, n: int = 16) -> np.ndarray:
    a = 2.0 * np.pi * np.arange(n) / n
    return np.stack([radius * np.cos(a), radius * np.sin(a)], 1).astype(np.float32)


def footprint_rect(length: float, width: float) -> np.ndarray:
    hl, hw = 0.5 * length, 0.5 * width
    return np.array([[-hl, -hw], [hl, -hw], [hl, hw], [-hl, hw]], np.float32)


def footprint_L(length=0.8, width=0.6, notch_l=0.4, notch_w=0.3) -> np.ndarray:
    """Nonconvex L: bounding box length x width with a notch_l x notch_w corner removed;
    6 corners + 6 edge midpoints = 12 ordered (CCW) vertices, collinear ones included."""
    hl, hw = 0.5 * length, 0.5 * width
    c = np.array([[-hl, -hw], [hl, -hw], [hl, hw - notch_w], [hl - notch_l, hw - notch_w],
                  [hl - notch_l, hw], [-hl, hw]], np.float64)
    out = []
    for k in range(6):
        out.append(c[k])
        out.append(0.5 * (c[k] + c[(k + 1) % 6]))
    return np.array(out, np.float32)


def beam_table(n_beams: int, fov_deg: float) -> np.ndarray:
    """FOV < 360: n_beams angles linearly spaced over [-FOV/2, +FOV/2] inclusive;
    360: -pi + j * 2 pi / n_beams."""
    if fov_deg >= 360.0:
        a = -np.pi + np.arange(n_beams) * (2.0 * np.pi / n_beams)
    else:
        half = np.deg2rad(fov_deg) / 2.0
        a = np.linspace(-half, half, n_beams)
    return a.astype(np.float32)


# ----------------------------------------------------------------------------- configs

def make_workload(cfg: int, n_envs: int | None = None) -> Workload:
    """cfg = 1..5 -> BASELINE.json configs[0..4]; 6 = the extra N-sweep workload of SURVEY.md 8(d)."""
    f32 = np.float32
    if cfg == 1:
        wl = Workload("C1-tiny", map_rectangles(256, 0.15, 0), RHO, footprint_ngon(0.2, 16),
                      beam_table(360, 360.0), f32(5.0), DRIVE_DIFF,
                      np.array([0, 1, 0, 0, -2, 2], f32), 64, f32(0.1), 100, 0)
    elif cfg == 2:
        wl = Workload("C2-rect-wheeled", map_rectangles(512, 0.20, 2, n_discs=30), RHO,
                      footprint_rect(0.6, 0.4), beam_table(720, 270.0), f32(10.0), DRIVE_DIFF,
                      np.array([-0.5, 1.5, 0, 0, -2.5, 2.5], f32), 4096, f32(0.1), 1000, 2)
    elif cfg == 3:
        wl = Workload("C3-nonconvex-omni", map_rectangles(512, 0.20, 3, n_discs=30), RHO,
                      footprint_L(), beam_table(360, 360.0), f32(8.0), DRIVE_OMNI,
                      np.array([-1, 1, -1, 1, -2, 2], f32), 8192, f32(0.05), 1000, 3)
    elif cfg == 4:
        wl = Workload("C4-large-narrow", map_large_maze(2048, 0.25, 4), RHO,
                      footprint_rect(0.5, 0.5), beam_table(128, 90.0), f32(6.0), DRIVE_DIFF,
                      np.array([-0.5, 1.5, 0, 0, -2.5, 2.5], f32), 16384, f32(0.1), 1000, 4,
                      forced_reset_frac=0.02)
    elif cfg == 5:
        occ, regions = map_tile_atlas(5)
        wl = Workload("C5-stress-tiles", occ, RHO, footprint_rect(0.5, 0.4),
                      beam_table(720, 270.0), f32(5.0), DRIVE_DIFF,
                      np.array([0, 1, 0, 0, -2, 2], f32), 65536, f32(0.1), 500, 5,
                      goal_dist_min=f32(1.0), goal_dist_max=f32(3.0), regions=regions,
                      ring_capacity=1 << 22)
    elif cfg == 6:
        # extra (context for PAPER.md:175 / Fig. 5): C1's robot on C2's map, for the N sweep
        wl = Workload("X-fig5-sweep", map_rectangles(512, 0.20, 2, n_discs=30), RHO, footprint_ngon(0.2, 16),
                      beam_table(360, 360.0), f32(5.0), DRIVE_DIFF,
                      np.array([0, 1, 0, 0, -2, 2], f32), 1024, f32(0.1), 1000, 6)
    else:
        raise ValueError("cfg must be 1..6")
    if n_envs is not None:
        wl.n_envs = int(n_envs)
    return wl


def tiny_workload(size=32, n_envs=8, n_beams=24, seed=7, drive=DRIVE_DIFF, footprint=None,
                  max_range=1.0, frac=0.12) -> Workload:
    """A small map for brute-force cross-checks (<= 32x32 cells)."""
    rng = np.random.default_rng(seed)
    occ = np.zeros((size, size), np.uint8)
    _border(occ)
    while occ.mean() < frac:
        _add_rect(occ, rng, 1, 5)  # tiny map: full mean is cheap
    lim = np.array([-0.5, 1.0, 0, 0, -2, 2], np.float32) if drive == DRIVE_DIFF else \
        np.array([-1, 1, -1, 1, -2, 2], np.float32)
    fp = footprint_rect(0.3, 0.2) if footprint is None else footprint
    return Workload(f"tiny{size}", occ, RHO, fp, beam_table(n_beams, 360.0),
                    np.float32(max_range), drive, lim, n_envs, np.float32(0.1), 10, seed,
                    goal_dist_min=np.float32(0.3), goal_dist_max=np.float32(1.0))


# ----------------------------------------------------------------------------- tapes

def action_tape(wl: Workload, steps: int, seed: int | None = None) -> np.ndarray:
    """float32 [steps, N, A] uniform within the velocity limits (physical units)."""
    rng = np.random.default_rng((wl.seed if seed is None else seed) + 1000)
    lim = wl.vel_limits.astype(np.float64)
    if wl.drive == DRIVE_DIFF:
        lo = np.array([lim[0], lim[4]])
        hi = np.array([lim[1], lim[5]])
    else:
        lo = np.array([lim[0], lim[2], lim[4]])
        hi = np.array([lim[1], lim[3], lim[5]])
    u = rng.random((steps, wl.n_envs, wl.action_dim), dtype=np.float32)
    return (lo.astype(np.float32) + u * (hi - lo).astype(np.float32)).astype(np.float32)


def seed_tape(wl: Workload, steps: int, seed: int | None = None) -> np.ndarray:
    """uint64 [steps, N]: one reset seed per env per step."""
    rng = np.random.default_rng((wl.seed if seed is None else seed) + 2000)
    return rng.integers(0, np.iinfo(np.uint64).max, size=(steps, wl.n_envs), dtype=np.uint64,
                        endpoint=True)


def forced_reset_tape(wl: Workload, steps: int, seed: int | None = None) -> np.ndarray:
    """uint8 [steps, N]: forced-reset requests (C4: a seeded random 2 % of envs each step)."""
    rng = np.random.default_rng((wl.seed if seed is None else seed) + 3000)
    if wl.forced_reset_frac <= 0.0:
        return np.zeros((steps, wl.n_envs), np.uint8)
    return (rng.random((steps, wl.n_envs)) < wl.forced_reset_frac).astype(np.uint8)


def random_poses(wl: Workload, n: int, seed: int) -> np.ndarray:
    """float32 [3, n]: x, y uniform over the map extent, psi uniform in [-pi, pi) (test inputs)."""
    rng = np.random.default_rng(seed + 4000)
    H, W = wl.occ.shape
    x = (rng.random(n) * W * float(wl.resolution)).astype(np.float32)
    y = (rng.random(n) * H * float(wl.resolution)).astype(np.float32)
    psi = (rng.random(n) * 2 * np.pi - np.pi).astype(np.float32)
    return np.stack([x, y, psi], 0)


def shard_envs(n_envs: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous env shard [lo, hi) of rank `rank` (envs are independent)."""
    base, rem = divmod(n_envs, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
