"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json `configs`).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: no quadrature, no basis functions, no Hamiltonian. It only places atoms and evaluates
analytic input fields (Gaussians, solid harmonics) at node coordinates that the caller obtained from
the library under test (`csf_node_coords` / `csf_mass_diag`, or the oracle's equivalents).

The synthetic systems stand in for the paper's twisted-bilayer WTe2 slabs and MnSi
supercells, whose structures and ONCV pseudopotentials are not available; only sizes
(DoF, electrons, order, boundary conditions) follow the paper.

Every random draw comes from numpy.random.Generator(PCG64(1000 + config index)) in the order:
atom positions, V depths, |B| magnitudes, B directions, channel widths per type, Delta per type, X.
"""
from dataclasses import dataclass, field
import numpy as np

BC_PERIODIC, BC_DIRICHLET = 0, 1
R_CUT_PROJ = 2.5      # bohr, hard cutoff of the projector radial functions (reading A10)
R_CUT_POT = 6.0       # bohr, truncation of the Gaussian potentials
N_CHANNELS = 6        # (l=0,tau=1) (l=0,tau=2) (l=1,j=1/2) (l=1,j=3/2) (l=2,j=3/2) (l=2,j=5/2)  (reading A9)
CHANNEL_L = (0, 0, 1, 1, 2, 2)
N_PROJ = sum(2 * l + 1 for l in CHANNEL_L)   # 18 scalar projector columns per atom


@dataclass(frozen=True)
class Config:
    index: int
    name: str
    ncell: tuple
    box: tuple
    order: int
    bc: tuple
    natoms: int
    placement: str
    nvec: int
    degree: int
    nstates: int = 0          # total spinor states of the system (blocks = ceil(nstates / nvec))
    seed: int = field(default=0)

    @property
    def nfree(self):
        return tuple(c * self.order - (1 if b == BC_DIRICHLET else 0) for c, b in zip(self.ncell, self.bc))

    @property
    def M(self):
        nx, ny, nz = self.nfree
        return nx * ny * nz


CONFIGS = {
    0: Config(0, "cfg0_tiny_periodic_p3", (3, 3, 3), (6.0, 6.0, 6.0), 3, (0, 0, 0), 2, "uniform", 16, 8, 16, 1000),
    1: Config(1, "cfg1_periodic_cube_p4", (10, 10, 10), (20.0, 20.0, 20.0), 4, (0, 0, 0), 32, "uniform_sep3", 256, 20, 256, 1001),
    2: Config(2, "cfg2_slab_p5", (20, 20, 40), (30.0, 30.0, 30.0), 5, (0, 0, 1), 200, "slab3", 512, 30, 5500, 1002),
    3: Config(3, "cfg3_bulk_p5", (32, 32, 32), (32.0, 32.0, 32.0), 5, (0, 0, 0), 500, "bcc_jitter", 256, 40, 7700, 1003),
    4: Config(4, "cfg4_large_p4", (40, 40, 40), (40.0, 40.0, 40.0), 4, (0, 0, 0), 1000, "rsa32", 256, 50, 22000, 1004),
}


def scaled_config(base: Config, ncell, natoms, nvec=None, degree=None, name=None) -> Config:
    """Same cell size, order and boundary conditions as `base` on a smaller mesh, atoms uniform with separation
    >= 3 bohr (parity sub-cases and the bounded CPU-baseline sample)."""
    h = [b / c for b, c in zip(base.box, base.ncell)]
    return Config(base.index, name or f"{base.name}_sub{ncell[0]}x{ncell[1]}x{ncell[2]}", tuple(ncell),
                  tuple(h[d] * ncell[d] for d in range(3)), base.order, base.bc, natoms, "uniform_sep3",
                  nvec or base.nvec, degree or base.degree, 0, base.seed)


def _min_image(d, L, periodic):
    return d - L * np.round(d / L) if periodic else d


def _separated(pos, cand, box, bc, dmin):
    if len(pos) == 0:
        return True
    d = np.asarray(pos) - cand
    for k in range(3):
        d[:, k] = _min_image(d[:, k], box[k], bc[k] == BC_PERIODIC)
    return bool(np.all(np.einsum("ij,ij->i", d, d) >= dmin * dmin))


def place_atoms(cfg: Config, rng) -> np.ndarray:
    box = np.asarray(cfg.box)
    if cfg.placement == "uniform":
        return rng.uniform(0.0, 1.0, (cfg.natoms, 3)) * box
    if cfg.placement in ("uniform_sep3", "rsa32"):
        dmin = 3.0 if cfg.placement == "uniform_sep3" else 3.2
        pos = []
        tries = 0
        while len(pos) < cfg.natoms:
            cand = rng.uniform(0.0, 1.0, 3) * box
            tries += 1
            if tries > 2000000:
                raise RuntimeError("atom placement did not converge")
            if _separated(pos, cand, cfg.box, cfg.bc, dmin):
                pos.append(cand)
        return np.asarray(pos)
    if cfg.placement == "slab3":
        # 3 layers, slab of 10 bohr centred in z with vacuum on both sides
        z0 = 0.5 * cfg.box[2] - 5.0
        layers = z0 + np.array([1.5, 5.0, 8.5])
        pos = []
        tries = 0
        while len(pos) < cfg.natoms:
            lay = len(pos) % 3
            cand = np.array([rng.uniform(0, cfg.box[0]), rng.uniform(0, cfg.box[1]), layers[lay] + rng.uniform(-0.5, 0.5)])
            tries += 1
            if tries > 2000000:
                raise RuntimeError("atom placement did not converge")
            if _separated(pos, cand, cfg.box, cfg.bc, 3.0):
                pos.append(cand)
        return np.asarray(pos)
    if cfg.placement == "bcc_jitter":
        k = 1
        while 2 * k ** 3 < cfg.natoms:
            k += 1
        g = np.stack(np.meshgrid(np.arange(k), np.arange(k), np.arange(k), indexing="ij"), -1).reshape(-1, 3).astype(float)
        sites = np.concatenate([g, g + 0.5]) / k
        pick = rng.choice(len(sites), cfg.natoms, replace=False)
        pos = sites[np.sort(pick)] * box + rng.uniform(-0.3, 0.3, (cfg.natoms, 3))
        return np.mod(pos, box)
    raise ValueError(cfg.placement)


def grid_axes(cfg: Config, coords: np.ndarray):
    """The three 1-D coordinate axes of the tensor-product node grid (x fastest numbering)."""
    nx, ny, nz = cfg.nfree
    assert coords.shape == (nx * ny * nz, 3)
    return coords[:nx, 0].copy(), coords[0:nx * ny:nx, 1].copy(), coords[0::nx * ny, 2].copy()


def _local_patch(cfg, axes, centre, rcut):
    """Indices and min-image displacements of the nodes within rcut of `centre`."""
    idx, disp = [], []
    for k in range(3):
        d = _min_image(axes[k] - centre[k], cfg.box[k], cfg.bc[k] == BC_PERIODIC)
        sel = np.nonzero(np.abs(d) <= rcut)[0]
        idx.append(sel); disp.append(d[sel])
    if min(len(s) for s in idx) == 0:
        return np.zeros(0, dtype=np.int64), np.zeros((0, 3))
    nx, ny, _ = cfg.nfree
    DZ, DY, DX = np.meshgrid(disp[2], disp[1], disp[0], indexing="ij")
    IZ, IY, IX = np.meshgrid(idx[2], idx[1], idx[0], indexing="ij")
    r2 = DX * DX + DY * DY + DZ * DZ
    m = r2 <= rcut * rcut
    node = (IX + nx * (IY + ny * IZ))[m].astype(np.int64)
    dxyz = np.stack([DX[m], DY[m], DZ[m]], -1)
    order = np.argsort(node, kind="stable")
    return node[order], dxyz[order]


def _solid_harmonics(l, d):
    """r^l Y_lm(r_hat), real form, m = -l..l, as polynomials in the displacement d[:, 3]."""
    x, y, z = d[:, 0], d[:, 1], d[:, 2]
    if l == 0:
        return np.full((len(d), 1), 0.5 / np.sqrt(np.pi))
    if l == 1:
        c = np.sqrt(3.0 / (4.0 * np.pi))
        return c * np.stack([y, z, x], -1)
    if l == 2:
        c = np.sqrt(15.0 / (4.0 * np.pi))
        r2 = x * x + y * y + z * z
        return np.stack([c * x * y, c * y * z, np.sqrt(5.0 / (16.0 * np.pi)) * (3.0 * z * z - r2), c * x * z, 0.5 * c * (x * x - y * y)], -1)
    raise ValueError(l)


@dataclass
class System:
    cfg: Config
    positions: np.ndarray
    veff: np.ndarray          # [M]
    bxyz: np.ndarray          # [M,3]
    node_ptr: np.ndarray      # [natoms+1] int64
    node_idx: np.ndarray      # int64 global node ids, sorted per atom
    nproj: np.ndarray         # [natoms] int32
    pvals: np.ndarray         # concatenated [n_a][nproj] row-major, entry = P_{I chi} (integrated, eq.42 at k=0)
    atom_type: np.ndarray     # [natoms] int32
    delta: np.ndarray         # concatenated per type [(2 npj)][(2 npj)] complex128, index 2 chi + alpha
    delta_ptr: np.ndarray     # [ntypes+1] int64
    delta_soc_off: np.ndarray # the SOC-off twin d (x) I_2 (same layout), for the SU(2) covariance check
    rng: object

    @property
    def coverage(self):
        """c_ov = sum_a n_a / M."""
        return float(self.node_ptr[-1]) / float(self.cfg.M)


def make_system(cfg: Config, coords: np.ndarray, mass: np.ndarray, with_projectors=True) -> System:
    """Atoms, V_eff, B, projectors and Delta for `cfg` at the node coordinates/lumped masses the library exported."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    axes = grid_axes(cfg, coords)
    M = cfg.M
    pos = place_atoms(cfg, rng)
    na = cfg.natoms
    depth = rng.uniform(-2.0, -0.5, na)
    bmag = rng.uniform(0.0, 0.3, na)
    nhat = rng.normal(size=(na, 3)); nhat /= np.linalg.norm(nhat, axis=1, keepdims=True)
    veff = np.zeros(M); bxyz = np.zeros((M, 3))
    for a in range(na):
        node, d = _local_patch(cfg, axes, pos[a], R_CUT_POT)
        g = np.exp(-0.5 * np.einsum("ij,ij->i", d, d))
        np.add.at(veff, node, depth[a] * g)
        for k in range(3):
            np.add.at(bxyz[:, k], node, bmag[a] * nhat[a, k] * g)
    ntypes = 2 if na > 1 else 1
    sigma = rng.uniform(0.5, 0.7, (ntypes, N_CHANNELS))
    npj2 = 2 * N_PROJ
    deltas, deltas_off = [], []
    for _ in range(ntypes):
        mag = rng.uniform(0.1, 1.0, (npj2, npj2)); ph = rng.uniform(0.0, 2.0 * np.pi, (npj2, npj2))
        A = mag * np.exp(1j * ph)
        D = np.triu(A, 1); D = D + D.conj().T + np.diag(rng.uniform(0.1, 1.0, npj2))
        deltas.append(D)
        d = np.abs(D[0::2, 0::2]); d = np.triu(d, 1); d = d + d.T + np.diag(np.real(np.diag(D))[0::2])
        deltas_off.append(np.kron(d, np.eye(2)).astype(np.complex128))
    delta = np.concatenate([D.reshape(-1) for D in deltas]); delta_off = np.concatenate([D.reshape(-1) for D in deltas_off])
    delta_ptr = np.arange(ntypes + 1, dtype=np.int64) * npj2 * npj2
    atom_type = (np.arange(na) % ntypes).astype(np.int32)
    node_ptr = np.zeros(na + 1, dtype=np.int64); idx_list, val_list = [], []
    if with_projectors:
        for a in range(na):
            node, d = _local_patch(cfg, axes, pos[a], R_CUT_PROJ)
            r2 = np.einsum("ij,ij->i", d, d)
            cols = []
            for ch, l in enumerate(CHANNEL_L):
                rad = np.exp(-0.5 * r2 / sigma[atom_type[a], ch] ** 2)
                cols.append(rad[:, None] * _solid_harmonics(l, d))
            P = np.concatenate(cols, 1) * mass[node][:, None]       # GLL collocation of eq.42: m_I p_chi(r_I - R_a)
            idx_list.append(node); val_list.append(P.reshape(-1)); node_ptr[a + 1] = node_ptr[a] + len(node)
        nproj = np.full(na, N_PROJ, dtype=np.int32)
        node_idx = np.concatenate(idx_list) if idx_list else np.zeros(0, dtype=np.int64)
        pvals = np.concatenate(val_list) if val_list else np.zeros(0)
    else:
        nproj = np.zeros(0, dtype=np.int32); node_idx = np.zeros(0, dtype=np.int64); pvals = np.zeros(0)
        atom_type = np.zeros(0, dtype=np.int32); node_ptr = np.zeros(1, dtype=np.int64)
    return System(cfg, pos, veff, bxyz, node_ptr, node_idx, nproj, pvals, atom_type, delta, delta_ptr, delta_off, rng)


def bloch_pvals(sysm: System, coords: np.ndarray, kvec) -> np.ndarray:
    """Complex projector entries P^{a,k}_{I chi} of eq.42 for Bloch vector k, same layout as `sysm.pvals`:
    the collocated entry m_I p_chi(r_I - L_q - R_a) times e^{-i k.(r_I - L_q)}, with r_I - L_q = R_a + d and d the
    minimum-image displacement the generator used for that support node (one image per node: r_c < L/2)."""
    cfg = sysm.cfg
    kvec = np.asarray(kvec, dtype=np.float64)
    axes = grid_axes(cfg, coords)
    out = np.zeros(sysm.pvals.size, dtype=np.complex128)
    off = 0
    for a in range(len(sysm.nproj)):
        node, d = _local_patch(cfg, axes, sysm.positions[a], R_CUT_PROJ)
        assert np.array_equal(node, sysm.node_idx[sysm.node_ptr[a]:sysm.node_ptr[a + 1]])
        npj = int(sysm.nproj[a])
        phase = np.exp(-1j * ((sysm.positions[a][None, :] + d) @ kvec))
        blk = sysm.pvals[off:off + node.size * npj].reshape(node.size, npj) * phase[:, None]
        out[off:off + node.size * npj] = blk.reshape(-1); off += node.size * npj
    return out


def random_block(rng, nrows, nvec) -> np.ndarray:
    """i.i.d. complex normal block, re and im ~ N(0, 1/2)."""
    return (rng.normal(scale=np.sqrt(0.5), size=(nrows, nvec)) + 1j * rng.normal(scale=np.sqrt(0.5), size=(nrows, nvec))).astype(np.complex128)
