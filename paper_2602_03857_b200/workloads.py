"""Seeded synthetic inputs for BASELINE.json's five configurations (recipe: DESIGN.md "Inputs").

This module serves BOTH the CUDA path and the CPU oracle and therefore holds NONE of the method's arithmetic:
it only lays out meshes, station sets, true density models and draws of standard-normal numbers.  Data
`d_obs = G m_true + sigma * noise` is formed by the caller with whichever forward operator it is testing.

The paper's own datasets (Sec. 4) are not available; these inputs stand in for them with the
same shapes: regular station grids over block / dyke models, irregular land stations over
topography, up to 3.3 M prisms and 178,797 stations.
"""
from dataclasses import dataclass, field

import numpy as np

GAMMA_MGAL = 6.674e-11 * 1e5      # mGal per (kg/m^3 * m): BASELINE.json config 1 ("G = 6.674e-11 SI", gz in mGal)
SEED0 = 26020385700                # seed = SEED0 + 10*cfg + stream
STREAM_MODEL, STREAM_XY, STREAM_TOPO, STREAM_NOISE, STREAM_VEC = 0, 1, 2, 3, 4


def rng(cfg: int, stream: int) -> np.random.Generator:
    return np.random.default_rng(SEED0 + 10 * cfg + stream)


@dataclass
class Workload:
    name: str
    cfg: int
    nx: int
    ny: int
    nz: int
    h: float
    xn: np.ndarray
    yn: np.ndarray
    zn: np.ndarray
    xo: np.ndarray
    yo: np.ndarray
    zo: np.ndarray
    m_true: np.ndarray          # kg/m^3, flat, cell (i,j,k) <-> (i*ny + j)*nz + k
    noise_frac: float           # sigma = noise_frac * max|G m_true|
    cg_iters: int
    beta: float = 2.0
    z0: float = 0.0
    gamma: float = GAMMA_MGAL
    lam_factor: float = 1e-2    # lambda = lam_factor * trace(G W^-2 G^T) / N
    extra: dict = field(default_factory=dict)

    @property
    def M(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def N(self) -> int:
        return int(self.xo.size)

    @property
    def n_nodes(self) -> int:
        return (self.nx + 1) * (self.ny + 1) * (self.nz + 1)

    def noise(self) -> np.ndarray:
        """Standard-normal draw for the data noise (scaled by the caller)."""
        return rng(self.cfg, STREAM_NOISE).standard_normal(self.N)

    def test_vectors(self):
        """(u_white[M], v_white[N], v_smooth[N]) for operator parity / timing."""
        g = rng(self.cfg, STREAM_VEC)
        u = g.standard_normal(self.M)
        v = g.standard_normal(self.N)
        cx, cy = 0.5 * (self.xn[0] + self.xn[-1]), 0.5 * (self.yn[0] + self.yn[-1])
        s = 0.2 * (self.xn[-1] - self.xn[0])
        vs = np.exp(-((self.xo - cx) ** 2 + (self.yo - cy) ** 2) / (2 * s * s))
        return u, v, vs


def _mesh(nx, ny, nz, h):
    return (np.arange(nx + 1, dtype=np.float64) * h, np.arange(ny + 1, dtype=np.float64) * h,
            np.arange(nz + 1, dtype=np.float64) * h)


def _grid_stations(nx, ny, h, height):
    xc = (np.arange(nx) + 0.5) * h
    yc = (np.arange(ny) + 0.5) * h
    X, Y = np.meshgrid(xc, yc, indexing="ij")       # station index i*ny + j
    return X.ravel().copy(), Y.ravel().copy(), np.full(nx * ny, -float(height))


def _topo(cfg, x, y, amp, lmin, lmax):
    g = rng(cfg, STREAM_TOPO)
    L = g.uniform(lmin, lmax, 8)
    th = g.uniform(0, 2 * np.pi, 8)
    ph = g.uniform(0, 2 * np.pi, 8)
    s = np.zeros_like(x)
    for t in range(8):
        s += np.sin(2 * np.pi * (x * np.cos(th[t]) + y * np.sin(th[t])) / L[t] + ph[t])
    s /= 8.0
    return amp * (1.0 + s) / 2.0                     # in [0, amp]: stations stay above the mesh top (reading C14)


def _box(m3, i0, i1, j0, j1, k0, k1, val, add=False):
    """Inclusive index ranges, clipped to the mesh."""
    nx, ny, nz = m3.shape
    sl = (slice(max(i0, 0), min(i1, nx - 1) + 1), slice(max(j0, 0), min(j1, ny - 1) + 1),
          slice(max(k0, 0), min(k1, nz - 1) + 1))
    if add:
        m3[sl] += val
    else:
        m3[sl] = val


def make(cfg: int) -> Workload:
    """BASELINE.json configs 1..5 (1-based), with SURVEY.md App. B's concrete choices; 6 = the paper's Table 1 shape."""
    if cfg == 1:
        nx, ny, nz, h = 16, 16, 8, 50.0
        xn, yn, zn = _mesh(nx, ny, nz, h)
        xo, yo, zo = _grid_stations(nx, ny, h, 1.0)
        m3 = np.zeros((nx, ny, nz))
        _box(m3, 6, 9, 6, 9, 2, 4, 500.0)           # reading C13
        return Workload("cfg1_tiny_block", 1, nx, ny, nz, h, xn, yn, zn, xo, yo, zo, m3.ravel(), 0.01, 50, z0=25.0)
    if cfg == 2:
        nx, ny, nz, h = 64, 64, 32, 25.0
        xn, yn, zn = _mesh(nx, ny, nz, h)
        xo, yo, zo = _grid_stations(nx, ny, h, 1.0)
        m3 = rng(2, STREAM_MODEL).standard_normal((nx, ny, nz)) * 10.0
        _box(m3, 31, 33, 12, 51, 2, 19, 300.0, add=True)
        return Workload("cfg2_vertical_dyke", 2, nx, ny, nz, h, xn, yn, zn, xo, yo, zo, m3.ravel(), 0.02, 100,
                        z0=h / 2)
    if cfg == 3:
        nx, ny, nz, h = 128, 128, 64, 20.0
        xn, yn, zn = _mesh(nx, ny, nz, h)
        xo, yo, zo = _grid_stations(nx, ny, h, 1.0)
        m3 = np.zeros((nx, ny, nz))
        for k in range(3, 50):
            i0 = 39 + (k - 3)
            _box(m3, i0, i0 + 3, 32, 95, k, k, 400.0)
        return Workload("cfg3_dipping_dyke", 3, nx, ny, nz, h, xn, yn, zn, xo, yo, zo, m3.ravel(), 0.02, 100,
                        z0=h / 2)
    if cfg == 4:
        nx, ny, nz, h = 200, 200, 50, 50.0
        xn, yn, zn = _mesh(nx, ny, nz, h)
        g = rng(4, STREAM_XY)
        N = 40000
        xo = g.uniform(0, nx * h, N)
        yo = g.uniform(0, ny * h, N)
        zo = -(_topo(4, xo, yo, 100.0, 2000.0, 10000.0) + 2.0)
        gm = rng(4, STREAM_MODEL)
        Lx, Ly, Lz = nx * h, ny * h, nz * h
        xc = (np.arange(nx) + 0.5) * h
        yc = (np.arange(ny) + 0.5) * h
        zc = (np.arange(nz) + 0.5) * h
        m3 = np.zeros((nx, ny, nz))
        for _ in range(6):
            cx, cy = gm.uniform(0.15, 0.85) * Lx, gm.uniform(0.15, 0.85) * Ly
            cz = gm.uniform(0.2, 0.7) * Lz
            ax, ay, az = gm.uniform(300, 1200), gm.uniform(300, 1200), gm.uniform(150, 500)
            drho = gm.choice([-1.0, 1.0]) * gm.uniform(200, 600)
            inside = (((xc[:, None, None] - cx) / ax) ** 2 + ((yc[None, :, None] - cy) / ay) ** 2 +
                      ((zc[None, None, :] - cz) / az) ** 2) <= 1.0
            m3[inside] += drho
        return Workload("cfg4_irregular_topo", 4, nx, ny, nz, h, xn, yn, zn, xo, yo, zo, m3.ravel(), 0.02, 100,
                        z0=h / 2)
    if cfg == 5:
        nx, ny, nz, h = 150, 148, 150, 100.0
        xn, yn, zn = _mesh(nx, ny, nz, h)
        g = rng(5, STREAM_XY)
        N = 178797
        xo = g.uniform(0, nx * h, N)
        yo = g.uniform(0, ny * h, N)
        zo = -(_topo(5, xo, yo, 200.0, 3000.0, 15000.0) + 1.0)
        m3 = rng(5, STREAM_MODEL).standard_normal((nx, ny, nz)) * 20.0
        dyke = np.zeros((nx, ny, nz), dtype=bool)
        dyke[40:43, 20:120, 2:60] = True                                    # V1
        dyke[30:130, 100:103, 3:50] = True                                  # V2
        for k in range(3, 60):                                               # D1 (dips along +x)
            i0 = 80 + (k - 3)
            dyke[max(i0, 0):min(i0 + 3, nx), 30:110, k] = True
        for k in range(5, 55):                                               # D2 (dips along -y)
            j0 = 70 - (k - 5)
            dyke[90:140, max(j0, 0):max(min(j0 + 3, ny), 0), k] = True
        m3[dyke] += 300.0
        return Workload("cfg5_largest", 5, nx, ny, nz, h, xn, yn, zn, xo, yo, zo, m3.ravel(), 0.02, 50, z0=h / 2)
    if cfg == 6:
        # Not a BASELINE.json config: the SHAPE of the paper's largest single-GPU benchmark (Table 1, P:168-178;
        # 2,601 stations x 3.28e6 cells, dense Float32 G = 34.13 GB), used by `bench.py --paper-shape` as the
        # one point of contact with the paper's own wall-clock numbers.  The paper's model is
        # not available; two +1000 kg/m^3 blocks stand in for its two-body synthetic.
        nx, ny, nz, h = 160, 160, 128, 100.0
        xn, yn, zn = _mesh(nx, ny, nz, h)
        ns = 51
        xs = (np.arange(ns) + 0.5) * (nx * h / ns)
        X, Y = np.meshgrid(xs, xs, indexing="ij")
        xo, yo, zo = X.ravel().copy(), Y.ravel().copy(), np.full(ns * ns, -1.0)
        m3 = np.zeros((nx, ny, nz))
        _box(m3, 40, 59, 60, 99, 10, 39, 1000.0)
        _box(m3, 100, 119, 60, 99, 20, 59, 1000.0)
        return Workload("paper_table1_shape", 6, nx, ny, nz, h, xn, yn, zn, xo, yo, zo, m3.ravel(), 0.01, 20,
                        z0=h / 2)
    raise ValueError(f"unknown config {cfg}")


def make_custom(nx, ny, nz, h, nobs, seed, topo_amp=0.0, clearance=1.0, rough=True, name=None) -> Workload:
    """A small workload of arbitrary shape for parity tests (ragged tiles, non-cubic cells, irregular stations).

    Node spacing is h in x, 0.8h in y and a mildly stretched spacing in z, so that nothing in the kernels can
    rely on cubic cells or uniform layers.  Stations are uniform random over the footprint (plus a margin),
    at `clearance` above a smooth topography of amplitude `topo_amp`.
    """
    g = np.random.default_rng(seed)
    xn = np.arange(nx + 1, dtype=np.float64) * h
    yn = np.arange(ny + 1, dtype=np.float64) * (0.8 * h)
    dz = h * (1.0 + 0.05 * np.arange(nz))
    zn = np.concatenate([[0.0], np.cumsum(dz)])
    Lx, Ly = xn[-1], yn[-1]
    xo = g.uniform(-0.1 * Lx, 1.1 * Lx, nobs)
    yo = g.uniform(-0.1 * Ly, 1.1 * Ly, nobs)
    topo = np.zeros(nobs)
    if topo_amp > 0:
        kx, ky, ph = g.uniform(1, 3, 3), g.uniform(1, 3, 3), g.uniform(0, 2 * np.pi, 3)
        s = sum(np.sin(2 * np.pi * (kx[t] * xo / Lx + ky[t] * yo / Ly) + ph[t]) for t in range(3)) / 3.0
        topo = topo_amp * (1 + s) / 2
    zo = -(topo + clearance)
    m = g.standard_normal(nx * ny * nz) * 50.0 if rough else np.ones(nx * ny * nz)
    cfg = 90 + (seed % 7)
    return Workload(name or f"custom_{nx}x{ny}x{nz}_{nobs}", cfg, nx, ny, nz, h, xn, yn, zn, xo, yo, zo, m, 0.02, 20,
                    z0=h / 2)
