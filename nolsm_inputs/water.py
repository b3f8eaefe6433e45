"""Water-like synthetic systems of BASELINE.json:configs[0..3] (recipe: DESIGN.md "Input recipe").

Stand-in for the CP2K H2O-dft-ls cell the paper measures on: 32-molecule cubic
cell of ~9.86 A (33.4 molecules/nm^3) replicated, block-sparse H and S with distance-decaying
elements and a spectral gap.  Output is a CSR-of-blocks store with uniform 6x6 blocks:
block k of row i holds the (i, col_idx[k]) block, row-major, FP32.

Only inputs are produced here; nothing of the NOLSM method itself.
"""
from dataclasses import dataclass
import numpy as np

from . import rng as _rng

GRID_PER_ANGSTROM = 65536          # positions, box and cutoff live on a 2^-16 A integer grid
BS = 6                             # basis functions per molecule: 4 (O-type site) + 1 + 1 (H-type sites)
N_OCC_PER_MOL = 4                  # occupied orbitals per molecule (closed shell)
N_ELEC_PER_MOL = 8                 # = 2 * N_OCC_PER_MOL
DENSITY = 0.0334                   # molecules per A^3
JITTER = 0.3                       # A, uniform per coordinate
SITE_OFFSETS = np.array([[0.0, 0.0, 0.0], [0.757, 0.586, 0.0], [-0.757, 0.586, 0.0]])  # A
ORB_SITE = np.array([0, 0, 0, 0, 1, 2])                     # orbital -> site within the molecule
ORB_ENERGY = np.array([-1.0, -1.0, -1.0, -1.0, -0.5, -0.5])  # Ha, on-site energies
S_AMPL, H_AMPL, H_LEN = 0.3, -0.2, 1.5
DEFAULT_SEED = 20210408

# name -> (n_mol, cutoff in A); BASELINE.json:configs[0..3]
CONFIGS = {
    "tiny32": (32, 6.0),
    "w4096": (4096, 8.0),
    "w32768": (32768, 10.0),
    "w262144": (262144, 12.0),
}


@dataclass
class WaterSystem:
    n_mol: int
    cutoff: float                  # A
    seed: int
    pos_q: np.ndarray              # [n_mol,3] int32, grid units, in [0, box_q)
    box_q: np.ndarray              # [3] int32, even
    rc_q: int                      # cutoff in grid units
    row_ptr: np.ndarray            # [n_mol+1] int32
    col_idx: np.ndarray            # [nnzb] int32, ascending within a row, self included
    h_val: np.ndarray              # [nnzb,6,6] float32
    s_val: np.ndarray              # [nnzb,6,6] float32
    n_electrons: float

    @property
    def nnzb(self):
        return int(self.col_idx.shape[0])

    @property
    def box_angstrom(self):
        return self.box_q.astype(np.float64) / GRID_PER_ANGSTROM


def _lattice(n_mol):
    """Lattice points in grid units and the (even) cubic box length."""
    k = round(n_mol ** (1.0 / 3.0))
    if k ** 3 == n_mol:
        a_q = 2 * int(round((1.0 / DENSITY) ** (1.0 / 3.0) * GRID_PER_ANGSTROM / 2.0))
        g = np.arange(k, dtype=np.int64)
        pts = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3) * a_q
        return pts, k * a_q
    c = round((n_mol / 4) ** (1.0 / 3.0))
    if 4 * c ** 3 != n_mol:
        raise ValueError("n_mol must be k^3 (simple cubic) or 4 c^3 (fcc)")
    a_q = 2 * int(round((4.0 / DENSITY) ** (1.0 / 3.0) * GRID_PER_ANGSTROM / 2.0))
    g = np.arange(c, dtype=np.int64)
    cells = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3) * a_q
    basis = np.array([[0, 0, 0], [1, 1, 0], [1, 0, 1], [0, 1, 1]], dtype=np.int64) * (a_q // 2)
    return (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3), c * a_q


def make_positions(n_mol, seed=DEFAULT_SEED):
    """Jittered lattice centres on the integer grid. Returns (pos_q int32 [n,3], box_q int32 [3])."""
    pts, box = _lattice(n_mol)
    jq = int(round(JITTER * GRID_PER_ANGSTROM))
    ctr = np.arange(n_mol * 3, dtype=np.uint64)
    jit = _rng.uniform_int(seed, 1, ctr, -jq, jq).reshape(n_mol, 3)
    pos = np.mod(pts + jit, box)
    return pos.astype(np.int32), np.array([box, box, box], dtype=np.int32)


def _pairs_bruteforce(pos, box, rc_q):
    n = pos.shape[0]
    rows, cols = [], []
    step = max(1, (1 << 22) // max(n, 1))
    p = pos.astype(np.int64)
    half = box.astype(np.int64) // 2
    for b in range(0, n, step):
        d = p[b:b + step, None, :] - p[None, :, :]
        d = np.where(d > half, d - box, d)
        d = np.where(d < -half, d + box, d)
        ok = (d * d).sum(-1) <= rc_q * rc_q
        r, c = np.nonzero(ok)
        rows.append(r + b)
        cols.append(c)
    return np.concatenate(rows), np.concatenate(cols)


def _pairs_kdtree(pos, box, rc_q):
    from scipy.spatial import cKDTree
    p = pos.astype(np.float64)
    tree = cKDTree(p, boxsize=box.astype(np.float64))
    cand = tree.query_ball_point(p, float(rc_q) + 2.0, workers=-1)
    cnt = np.fromiter((len(c) for c in cand), dtype=np.int64, count=len(cand))
    rows = np.repeat(np.arange(len(cand), dtype=np.int64), cnt)
    cols = np.concatenate([np.asarray(c, dtype=np.int64) for c in cand])
    pi = pos.astype(np.int64)
    half = box.astype(np.int64) // 2
    d = pi[rows] - pi[cols]
    d = np.where(d > half, d - box, d)
    d = np.where(d < -half, d + box, d)
    ok = (d * d).sum(-1) <= rc_q * rc_q
    return rows[ok], cols[ok]


def _pattern(pos, box, rc_q):
    n = pos.shape[0]
    if n <= 2048 or 2 * (rc_q + 2) >= int(box.min()):
        r, c = _pairs_bruteforce(pos, box, rc_q)
    else:
        r, c = _pairs_kdtree(pos, box, rc_q)
    order = np.lexsort((c, r))
    r, c = r[order], c[order]
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    np.add.at(row_ptr, r + 1, 1)
    return np.cumsum(row_ptr).astype(np.int32), r.astype(np.int32), c.astype(np.int32)


def _blocks(pos, box, rows, cols, chunk=1 << 18):
    """6x6 H and S blocks for molecule pairs (rows[k], cols[k])."""
    nnzb = rows.shape[0]
    h = np.empty((nnzb, BS, BS), dtype=np.float32)
    s = np.empty((nnzb, BS, BS), dtype=np.float32)
    inv = 1.0 / GRID_PER_ANGSTROM
    L = box.astype(np.float64) * inv
    same_site = ORB_SITE[:, None] == ORB_SITE[None, :]
    eye = np.eye(BS, dtype=bool)
    for b in range(0, nnzb, chunk):
        ri, ci = rows[b:b + chunk], cols[b:b + chunk]
        ctr = (pos[ri].astype(np.float64) - pos[ci].astype(np.float64)) * inv          # [m,3]
        d = ctr[:, None, None, :] + SITE_OFFSETS[None, :, None, :] - SITE_OFFSETS[None, None, :, :]
        d -= L * np.rint(d / L)
        r2 = (d * d).sum(-1)                                                             # [m,3,3]
        s_site = S_AMPL * np.exp(-0.5 * r2)
        h_site = H_AMPL * np.exp(-np.sqrt(r2) / H_LEN)
        sb = s_site[:, ORB_SITE[:, None], ORB_SITE[None, :]]
        hb = h_site[:, ORB_SITE[:, None], ORB_SITE[None, :]]
        self_pair = (ri == ci)
        if self_pair.any():
            sb[self_pair] = np.where(same_site, 0.0, sb[self_pair])
            hb[self_pair] = np.where(same_site, 0.0, hb[self_pair])
            sb[self_pair] = np.where(eye, 1.0, sb[self_pair])
            hb[self_pair] = np.where(eye, ORB_ENERGY[:, None] * np.ones((1, BS)), hb[self_pair])
        s[b:b + chunk] = sb.astype(np.float32)
        h[b:b + chunk] = hb.astype(np.float32)
    return h, s


def make_water_system(n_mol, cutoff, seed=DEFAULT_SEED):
    """Positions, neighbour pattern (centre distance <= cutoff, min image, closed ball, self
    included) and FP32 H, S blocks.  H and S share one pattern; both are zero outside it."""
    pos, box = make_positions(n_mol, seed)
    rc_q = int(round(cutoff * GRID_PER_ANGSTROM))
    row_ptr, rows, cols = _pattern(pos, box, rc_q)
    h, s = _blocks(pos, box, rows, cols)
    return WaterSystem(n_mol=n_mol, cutoff=float(cutoff), seed=seed, pos_q=pos, box_q=box, rc_q=rc_q,
                       row_ptr=row_ptr, col_idx=cols, h_val=h, s_val=s,
                       n_electrons=float(N_ELEC_PER_MOL * n_mol))


def model_parameters(system):
    """The constants of the element model above (the recipe of `_blocks`), for consumers that evaluate
    the elements themselves (nolsm.h: nolsm_model).  Values only; the positions stay in `system`."""
    return dict(box_q=[int(x) for x in system.box_q], rc_q=int(system.rc_q),
                unit_per_grid=1.0 / GRID_PER_ANGSTROM, site_offset=SITE_OFFSETS.tolist(),
                orb_site=ORB_SITE.tolist(), orb_energy=ORB_ENERGY.tolist(),
                s_ampl=S_AMPL, h_ampl=H_AMPL, h_len=H_LEN)


def to_dense(system, which):
    """Assemble the full (6 n_mol)^2 FP64 matrix from the block store (tests only; small systems)."""
    val = system.h_val if which == "H" else system.s_val
    n = system.n_mol * BS
    out = np.zeros((n, n))
    for i in range(system.n_mol):
        for k in range(system.row_ptr[i], system.row_ptr[i + 1]):
            j = system.col_idx[k]
            out[i * BS:(i + 1) * BS, j * BS:(j + 1) * BS] = val[k]
    return out
