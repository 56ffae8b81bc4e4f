"""Seeded synthetic INPUTS shared by the CUDA path, the oracle, the tests and bench.py.

This module holds none of the method's arithmetic (no ray generation, no sampling, no
compositing, no noise hashing, no source evaluation).  It only *describes* inputs: cube shapes,
camera matrices, transfer-function tables and seeded source-parameter lists.  Both the CUDA
library (`libvr`) and the CPU oracle (`oracle/`) consume exactly these arrays.

Stand-ins: the paper's cubes (HIPASS 1721x1721x1025 float32, PAPER.md line 57 footnote 4; the
Ursa Major HI cube, Fig. 1) are not available, so the recipes below follow
BASELINE.json `configs[0..4]` and SURVEY.md section 8(d).  Units are noise sigma.

Matrix convention: 4x4, row-major, column vectors, clip = M . (x, y, z, 1)^T
with (x, y, z) in voxel-index coordinates (RA, Dec, frequency), OpenGL clip space (NDC in
[-1, 1]^3, z = -1 near, +1 far).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 0x10122909          # cube seed = SEED_BASE + config index
VIEW_XOR = 0xA5A5               # view seed = cube seed ^ VIEW_XOR

# columns of a source row (float64): see `make_sources`
SRC_COLS = 16
(S_X0, S_Y0, S_Z0, S_AMP, S_SA, S_SB, S_SZ, S_COS, S_SIN, S_GRAD,
 S_XLO, S_XHI, S_YLO, S_YHI, S_ZLO, S_ZHI) = range(SRC_COLS)


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config (or a small test variant of it)."""
    name: str
    index: int                      # BASELINE.json configs[] index (seed offset)
    dims: tuple                     # (NX, NY, NZ) = (RA, Dec, freq), x fastest
    brick: tuple                    # configured brick size (BX, BY, BZ)
    frame: tuple                    # (W, H) of the full frame
    step: float                     # sampling step, voxels
    n_sources: int
    kind: str = "hi"                # "simple" (C1 recipe) or "hi" (C2..C5 recipe)
    continuum: float = 0.0          # + continuum * z / (NZ - 1)
    zero_fraction: float = 0.0      # fraction of configured bricks that are all-zero
    projection: str = "perspective"
    panels: tuple = (1, 1)          # tiled-display split of the frame (cols, rows)
    tf: str = "src"
    tau: float = 0.99               # ERT threshold (> 1 disables)
    notes: str = ""

    @property
    def seed(self) -> int:
        return SEED_BASE + self.index

    @property
    def view_seed(self) -> int:
        return self.seed ^ VIEW_XOR

    @property
    def n_voxels(self) -> int:
        return self.dims[0] * self.dims[1] * self.dims[2]

    @property
    def brick_grid(self) -> tuple:
        return tuple(-(-n // b) for n, b in zip(self.dims, self.brick))


# BASELINE.json configs[0..4]  (SURVEY.md 8(a) sizes)
C1 = Workload("C1", 0, (64, 64, 64), (64, 64, 64), (256, 256), 0.5, 3, kind="simple",
              projection="orthographic", tf="ramp", tau=2.0)
C2 = Workload("C2", 1, (512, 512, 1024), (64, 64, 64), (1920, 1080), 0.5, 200)
C3 = Workload("C3", 2, (2048, 2048, 4096), (256, 256, 256), (1920, 1080), 0.5, 20000,
              continuum=2.0, notes="360-frame orbit, MIP and EA")
C4 = Workload("C4", 3, (1024, 1024, 2048), (128, 128, 128), (9600, 5400), 0.25, 2000,
              panels=(5, 5))
C5 = Workload("C5", 4, (4096, 4096, 2048), (256, 256, 256), (9600, 5400), 0.5, 80000,
              zero_fraction=0.1, panels=(5, 5))
# Beyond BASELINE.json's five: the shape of the paper's largest rendered cube (HIPASS:
# 1721 x 1721 x 1025, "12 GB", shown at 3000 x 3000 and 8000 x 8000, line 61; partial edge bricks on every face), and a
# 256 GiB-class cube (as float32; "larger than a single machine memory limit", line 47 towards WALLABY)
# that fits one B200 only with float16 voxels.  Same recipe as C3.
HIPASS = Workload("HIPASS", 5, (1721, 1721, 1025), (256, 256, 256), (3000, 3000), 0.5, 3000, continuum=2.0,
                  notes="PAPER.md line 57 shape, synthetic content")
W256 = Workload("W256", 6, (4096, 4096, 4096), (256, 256, 256), (1920, 1080), 0.5, 160000, continuum=2.0,
                notes="256 GiB as float32: resident as float16 only")
CONFIGS = {w.name: w for w in (C1, C2, C3, C4, C5, HIPASS, W256)}


def scaled(w: Workload, name: str, dims, brick, frame, n_sources=None, panels=None) -> Workload:
    """A small test-sized variant of a config with the same recipe and seed."""
    from dataclasses import replace
    return replace(w, name=name, dims=tuple(dims), brick=tuple(brick), frame=tuple(frame),
                   n_sources=w.n_sources if n_sources is None else n_sources,
                   panels=w.panels if panels is None else tuple(panels))


# --------------------------------------------------------------------------------------
# sources (parameters only; the evaluation formula lives in oracle/ and in the CUDA generator)
# --------------------------------------------------------------------------------------
def make_sources(w: Workload) -> np.ndarray:
    """Seeded source-parameter table, float64 [n_sources, SRC_COLS].

    Row = (x0, y0, z0, amplitude, sigma_a, sigma_b, sigma_z, cos(theta), sin(theta), gradient,
    xlo, xhi, ylo, yhi, zlo, zhi).  The last six are the *integer* inclusive bounding box (clipped
    to the cube) outside which the source contributes nothing: the "truncated at 4 sigma" of
    SURVEY.md 8(d), made an integer input so that no floating-point knife-edge decides it.
    Recipes: SURVEY.md 8(d) bullet "Source s".
    """
    rng = np.random.Generator(np.random.PCG64(w.seed))
    n = w.n_sources
    nx, ny, nz = w.dims
    out = np.zeros((n, SRC_COLS), dtype=np.float64)
    if n == 0:
        return out
    if w.kind == "simple":          # C1: amplitude 5-20, per-axis sigma 2-6, no rotation/gradient
        amp = rng.uniform(5.0, 20.0, n)
        sa = rng.uniform(2.0, 6.0, n)
        sb = rng.uniform(2.0, 6.0, n)
        sz = rng.uniform(2.0, 6.0, n)
        theta = np.zeros(n)
        grad = np.zeros(n)
    else:                           # C2..C5: HI-like ellipsoidal Gaussians with velocity gradient
        amp = np.exp(rng.uniform(math.log(3.0), math.log(30.0), n))   # peak SNR log-uniform
        s1 = rng.uniform(2.0, 10.0, n)
        s2 = rng.uniform(2.0, 10.0, n)
        sa, sb = np.maximum(s1, s2), np.minimum(s1, s2)               # a = major axis
        theta = rng.uniform(0.0, math.pi, n)
        fwhm = rng.uniform(10.0, 60.0, n)
        sz = fwhm / 2.3548
        grad = rng.uniform(-1.0, 1.0, n) * fwhm / (4.0 * sa)
    hx = np.ceil(4.0 * np.maximum(sa, sb))
    hy = hx.copy()
    hz = np.ceil(4.0 * sz + np.abs(grad) * 4.0 * sa)
    # centres at least 4 sigma (of the smallest spatial sigma) from the faces where possible
    def centre(nn, margin):
        lo = np.minimum(margin, (nn - 1) / 2.0)
        return lo + rng.uniform(0.0, 1.0, n) * ((nn - 1) - 2.0 * lo)
    x0 = centre(nx, 4.0 * sb)
    y0 = centre(ny, 4.0 * sb)
    z0 = centre(nz, np.minimum(4.0 * sz, nz / 4.0))
    out[:, S_X0], out[:, S_Y0], out[:, S_Z0] = x0, y0, z0
    out[:, S_AMP], out[:, S_SA], out[:, S_SB], out[:, S_SZ] = amp, sa, sb, sz
    out[:, S_COS], out[:, S_SIN], out[:, S_GRAD] = np.cos(theta), np.sin(theta), grad
    out[:, S_XLO] = np.clip(np.floor(x0 - hx), 0, nx - 1)
    out[:, S_XHI] = np.clip(np.ceil(x0 + hx), 0, nx - 1)
    out[:, S_YLO] = np.clip(np.floor(y0 - hy), 0, ny - 1)
    out[:, S_YHI] = np.clip(np.ceil(y0 + hy), 0, ny - 1)
    out[:, S_ZLO] = np.clip(np.floor(z0 - hz), 0, nz - 1)
    out[:, S_ZHI] = np.clip(np.ceil(z0 + hz), 0, nz - 1)
    return out


def make_zero_boxes(w: Workload) -> np.ndarray:
    """int32 [n, 6] inclusive voxel boxes (xlo, xhi, ylo, yhi, zlo, zhi) that are all-zero
    ("flagged channels", BASELINE.json configs[4]): floor(zero_fraction * n_bricks) configured
    bricks chosen by a seeded shuffle."""
    gx, gy, gz = w.brick_grid
    nb = gx * gy * gz
    n = int(math.floor(w.zero_fraction * nb))
    if n == 0:
        return np.zeros((0, 6), dtype=np.int32)
    rng = np.random.Generator(np.random.PCG64(w.seed ^ 0x5EED))
    ids = np.sort(rng.permutation(nb)[:n])
    bx, by, bz = w.brick
    nx, ny, nz = w.dims
    out = np.zeros((n, 6), dtype=np.int32)
    for r, b in enumerate(ids):
        ix, iy, iz = b % gx, (b // gx) % gy, b // (gx * gy)
        out[r] = (ix * bx, min((ix + 1) * bx, nx) - 1, iy * by, min((iy + 1) * by, ny) - 1,
                  iz * bz, min((iz + 1) * bz, nz) - 1)
    return out


# --------------------------------------------------------------------------------------
# transfer functions (tables only; lookup + opacity correction are the method's)
# --------------------------------------------------------------------------------------
def _colour_ramp() -> np.ndarray:
    i = np.arange(256, dtype=np.float64) / 255.0
    t = np.zeros((256, 4), dtype=np.float64)
    t[:, 0] = i
    t[:, 1] = 1.0 - np.abs(2.0 * i - 1.0)
    t[:, 2] = 1.0 - i
    return t


def tf_ramp():
    """TF-ramp (C1, "linear-ramp"): vmin 0, vmax 20, alpha_i = 0.5 i/255 per voxel length."""
    t = _colour_ramp()
    t[:, 3] = 0.5 * np.arange(256) / 255.0
    return t.astype(np.float32), 0.0, 20.0


def tf_src(threshold: int = 32):
    """TF-src (C2..C5): vmin 0, vmax 32, alpha 0 for i <= threshold (32: v <= 4.02 sigma, noise is
    transparent), then linear to 0.25 at i = 255.  Other thresholds model the astronomer dragging
    the opacity threshold of the colour map (bench.py's tf_edit_ms)."""
    t = _colour_ramp()
    i = np.arange(256, dtype=np.float64)
    t[:, 3] = np.where(i <= threshold, 0.0, 0.25 * (i - threshold) / (255.0 - threshold))
    return t.astype(np.float32), 0.0, 32.0


def tf_fog():
    """TF-fog (stress variant): as TF-src but the alpha ramp starts at i = 0."""
    t = _colour_ramp()
    t[:, 3] = 0.25 * np.arange(256) / 255.0
    return t.astype(np.float32), 0.0, 32.0


TFS = {"ramp": tf_ramp, "src": tf_src, "fog": tf_fog}


# --------------------------------------------------------------------------------------
# cameras (4x4 matrices as inputs; how rays are derived from them is the method's)
# --------------------------------------------------------------------------------------
def _look_at(eye, centre, up):
    f = centre - eye
    f = f / np.linalg.norm(f)
    s = np.cross(f, up)
    s = s / np.linalg.norm(s)
    u = np.cross(s, f)
    V = np.eye(4)
    V[0, :3], V[1, :3], V[2, :3] = s, u, -f
    V[:3, 3] = -V[:3, :3] @ eye
    return V


def _frustum(l, r, b, t, n, f):
    P = np.zeros((4, 4))
    P[0, 0] = 2 * n / (r - l); P[0, 2] = (r + l) / (r - l)
    P[1, 1] = 2 * n / (t - b); P[1, 2] = (t + b) / (t - b)
    P[2, 2] = -(f + n) / (f - n); P[2, 3] = -2 * f * n / (f - n)
    P[3, 2] = -1.0
    return P


def _ortho(l, r, b, t, n, f):
    P = np.eye(4)
    P[0, 0] = 2 / (r - l); P[0, 3] = -(r + l) / (r - l)
    P[1, 1] = 2 / (t - b); P[1, 3] = -(t + b) / (t - b)
    P[2, 2] = -2 / (f - n); P[2, 3] = -(f + n) / (f - n)
    return P


def _centre_radius(dims):
    n1 = np.array(dims, dtype=np.float64) - 1.0
    return n1 / 2.0, 0.5 * float(np.linalg.norm(n1))


def _eye_dir(az_deg, el_deg):
    az, el = math.radians(az_deg), math.radians(el_deg)
    # up = +y (Dec); azimuth rotates about y starting from +z (frequency axis)
    return np.array([math.cos(el) * math.sin(az), math.sin(el), math.cos(el) * math.cos(az)])


def perspective_camera(dims, frame, azimuth_deg=30.0, elevation_deg=20.0, fovy_deg=40.0):
    """SURVEY.md 8(d) camera: centre c = (N-1)/2, R = |N-1|/2, distance 1.05 R / sin(fovy/2),
    near/far = distance -/+ 1.05 R, up +y, OpenGL-style M = P . V (model = identity)."""
    c, R = _centre_radius(dims)
    W, H = frame
    half = math.radians(fovy_deg) / 2.0
    dist = 1.05 * R / math.sin(half)
    near, far = dist - 1.05 * R, dist + 1.05 * R
    eye = c + dist * _eye_dir(azimuth_deg, elevation_deg)
    V = _look_at(eye, c, np.array([0.0, 1.0, 0.0]))
    top = near * math.tan(half)
    right = top * W / H
    return (_frustum(-right, right, -top, top, near, far) @ V).astype(np.float32)


def ortho_camera(dims, frame, direction, half_height=None):
    """Orthographic view along `direction` (from the camera towards the cube), half-height
    1.05 R by default."""
    c, R = _centre_radius(dims)
    W, H = frame
    d = np.asarray(direction, dtype=np.float64)
    d = d / np.linalg.norm(d)
    hh = 1.05 * R if half_height is None else half_height
    hw = hh * W / H
    up = np.array([0.0, 1.0, 0.0]) if abs(d[1]) < 0.9 else np.array([0.0, 0.0, 1.0])
    eye = c - d * (2.0 * R)
    V = _look_at(eye, c, up)
    return (_ortho(-hw, hw, -hh, hh, 2.0 * R - 1.05 * R, 2.0 * R + 1.05 * R) @ V).astype(np.float32)


def seeded_directions(seed: int, n: int = 3) -> np.ndarray:
    """n directions uniform on the sphere from the view seed (C1's "3 seeded view angles")."""
    rng = np.random.Generator(np.random.PCG64(seed))
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def axis_ortho_camera(dims, axis: int, sign: int = +1, near_offset: float = 8.0):
    """Axis-aligned orthographic view whose rays pass exactly through voxel centres: one pixel
    per voxel column, the box [-1/2, P-1/2] of the two screen axes mapped to NDC with P the next
    power of two >= N (pixels >= N miss the cube), near plane `near_offset` voxels in front of
    the entry face (a whole multiple of the step), everything dyadic so that positions are exact
    in float32 (SURVEY.md 8(c) pins for O-2/O-3/O-5).
    Returns (matrix float32, (W, H)).  `axis` is the marching axis, `sign` its direction."""
    N = list(dims)
    ua, va = [(1, 2), (0, 2), (0, 1)][axis]          # screen x axis, screen y axis (row 0 on top)
    W, H = (int(2 ** math.ceil(math.log2(N[ua]))), int(2 ** math.ceil(math.log2(N[va]))))
    M = np.zeros((4, 4))
    # xn = 2 (u + 1/2) / W - 1 ;  yn = 1 - 2 (v + 1/2) / H  (pixel j <-> voxel v = j)
    M[0, ua] = 2.0 / W; M[0, 3] = 1.0 / W - 1.0
    M[1, va] = -2.0 / H; M[1, 3] = 1.0 - 1.0 / H
    depth = N[axis] - 1 + 2.0 * near_offset
    depth = float(2 ** math.ceil(math.log2(depth)))     # dyadic depth range
    if sign > 0:      # march towards +axis: near plane at -near_offset
        M[2, axis] = 2.0 / depth; M[2, 3] = 2.0 * near_offset / depth - 1.0
    else:             # march towards -axis: near plane at N-1+near_offset
        M[2, axis] = -2.0 / depth; M[2, 3] = 2.0 * (N[axis] - 1 + near_offset) / depth - 1.0
    M[3, 3] = 1.0
    return M.astype(np.float32), (W, H)


def panel_matrix(M: np.ndarray, cols: int, rows: int, c: int, r: int) -> np.ndarray:
    """Off-axis sub-frustum (c, r) of a cols x rows split of the camera M (PAPER.md line 37,
    5 x 5 screens; BASELINE.json configs[3]): the NDC window of panel (c, r), row 0 on top, is
    stretched to [-1, 1]^2 by a clip-space scale + shear, so near and far planes are shared."""
    S = np.eye(4)
    S[0, 0] = cols; S[0, 3] = cols - 1 - 2 * c
    S[1, 1] = rows; S[1, 3] = -(rows - 1 - 2 * r)
    return (S @ M.astype(np.float64)).astype(np.float32)


def config_camera(w: Workload, frame_index: int = 0, frame=None) -> np.ndarray:
    """The camera BASELINE.json's config asks for (C3: azimuth = frame index in degrees)."""
    frame = w.frame if frame is None else frame
    if w.projection == "orthographic":
        d = seeded_directions(w.view_seed, 3)[frame_index % 3]
        return ortho_camera(w.dims, frame, d)
    az = float(frame_index) if w.name.startswith(("C3", "W256")) else 30.0 + float(frame_index)
    return perspective_camera(w.dims, frame, azimuth_deg=az)
