"""Seeded synthetic input generators for the five BASELINE.json workloads.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path.  It
holds none of the method's arithmetic: it only draws geometries, exponents,
normalisation constants, density-matrix factors and potentials from a seeded
``numpy.random.default_rng`` and packs them in the flat arrays the C ABI of
``include/gpw.h`` takes (cell, atoms, shells, primitive exponents and
coefficients, meshes).  The recipe is stated in DESIGN.md ("Input recipe") and
follows SURVEY.md section 8(d); the paper's own workloads (CP2K
water boxes, ASE diamond supercells, GTH basis sets) are not available, these
stand in for them with the same shapes.

It imports neither ``oracle`` nor the CUDA binding.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Sequence

import numpy as np

BASE_SEED = 20260324


def ncart(l: int) -> int:
    """Number of Cartesian components of a shell of angular momentum l."""
    return (l + 1) * (l + 2) // 2


def cart_powers(l: int):
    """(lx, ly, lz) of every Cartesian component, lexicographic with
    decreasing lx then decreasing ly (reading A2)."""
    out = []
    for lx in range(l, -1, -1):
        for ly in range(l - lx, -1, -1):
            out.append((lx, ly, l - lx - ly))
    return out


def _dfact(n: int) -> float:
    r = 1.0
    while n > 1:
        r *= n
        n -= 2
    return r


def gto_norm(l: int, a: float) -> float:
    """Caller-side normalisation (reading A1): x^l exp(-a r^2) has
    unit self-overlap in free space; shared by all components of the shell."""
    return math.sqrt((2.0 * a / math.pi) ** 1.5 * (4.0 * a) ** l / _dfact(2 * l - 1))


@dataclasses.dataclass
class GPWInputs:
    name: str
    cell: np.ndarray            # (3,3) rows = lattice vectors, Bohr
    xyz: np.ndarray             # (natm,3) Bohr
    shl_atom: np.ndarray        # (nshl,) int32
    shl_l: np.ndarray           # (nshl,) int32
    shl_nprim: np.ndarray       # (nshl,) int32
    shl_prim_off: np.ndarray    # (nshl,) int32
    prim_exp: np.ndarray        # (nprim,) float64
    prim_coef: np.ndarray       # (nprim,) float64
    mesh: np.ndarray            # (nlevel,3) int32, finest first
    tau: float
    rel_cutoff: float
    hermi: int
    deriv: int
    C: np.ndarray               # (nao,nocc): D = C C^T
    seed: int
    v_const: Optional[float] = None   # if set, v == this constant (tests)

    @property
    def natm(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def nshl(self) -> int:
        return int(self.shl_l.shape[0])

    @property
    def nlevel(self) -> int:
        return int(self.mesh.shape[0])

    @property
    def ao_loc(self) -> np.ndarray:
        n = np.array([ncart(int(l)) for l in self.shl_l], dtype=np.int64)
        return np.concatenate([[0], np.cumsum(n)])

    @property
    def nao(self) -> int:
        return int(self.ao_loc[-1])

    @property
    def ncomp(self) -> int:
        """Grid components: value | value + gradient | value + gradient + kinetic-energy density."""
        return {0: 1, 1: 4, 2: 5}[int(self.deriv)]

    def D(self) -> np.ndarray:
        return np.ascontiguousarray(self.C @ self.C.T)

    def D_block(self, rows: slice, cols: slice) -> np.ndarray:
        return self.C[rows] @ self.C[cols].T

    def v(self, level: int, ncomp: Optional[int] = None) -> np.ndarray:
        """Potential on one level: independent N(0,1) per point and component
        (reading A19).  Shape [ncomp, N1, N2, N3]."""
        nc = self.ncomp if ncomp is None else ncomp
        n1, n2, n3 = (int(x) for x in self.mesh[level])
        if self.v_const is not None:
            out = np.zeros((nc, n1, n2, n3))
            out[0] = self.v_const
            return out
        rng = np.random.default_rng([self.seed, 7000 + level])
        out = rng.standard_normal((4, n1, n2, n3))[:nc].copy()
        if nc == 5:   # the meta-GGA component has its own stream, so that components 0..3 do not depend on deriv
            rng5 = np.random.default_rng([self.seed, 9000 + level])
            out = np.concatenate([out, rng5.standard_normal((1, n1, n2, n3))])
        return out

    def abi_args(self):
        """Positional arguments of gpw_build_pairs up to (and excluding) plan_out."""
        return (self.cell, self.natm, self.xyz, self.nshl, self.shl_atom,
                self.shl_l, self.shl_nprim, self.shl_prim_off, self.prim_exp,
                self.prim_coef, self.nlevel, self.mesh, self.tau,
                self.rel_cutoff, self.hermi)


def pack_shells(atom_shells: Sequence[Sequence[tuple]]):
    """atom_shells[iatm] = [(l, [exps], [coefs]), ...] -> flat ABI arrays."""
    shl_atom, shl_l, shl_nprim, shl_off, pe, pc = [], [], [], [], [], []
    for ia, shells in enumerate(atom_shells):
        for (l, exps, coefs) in shells:
            shl_atom.append(ia)
            shl_l.append(l)
            shl_nprim.append(len(exps))
            shl_off.append(len(pe))
            pe.extend(float(e) for e in exps)
            pc.extend(float(c) for c in coefs)
    return (np.array(shl_atom, np.int32), np.array(shl_l, np.int32),
            np.array(shl_nprim, np.int32), np.array(shl_off, np.int32),
            np.array(pe, np.float64), np.array(pc, np.float64))


def _loguniform(rng, lo, hi, n):
    return np.exp(rng.uniform(math.log(lo), math.log(hi), n))


def _single_prim_shells(ls, exps):
    return [(int(l), [float(a)], [gto_norm(int(l), float(a))]) for l, a in zip(ls, exps)]


def _water_geometry(rng, nmol: int, edge: float, oo_min: float = 4.8):
    """Rigid waters (O-H 1.81 Bohr, HOH 104.5 deg), uniform random position and
    orientation, rejecting minimum-image O-O distances below oo_min."""
    roh, ang = 1.81, math.radians(104.5)
    h1 = np.array([roh * math.sin(ang / 2), roh * math.cos(ang / 2), 0.0])
    h2 = np.array([-roh * math.sin(ang / 2), roh * math.cos(ang / 2), 0.0])
    opos = np.zeros((0, 3))
    xyz = []
    tries = 0
    while opos.shape[0] < nmol:
        tries += 1
        if tries > 5_000_000:
            raise RuntimeError("water insertion did not converge")
        o = rng.uniform(0.0, edge, 3)
        if opos.shape[0]:
            d = opos - o
            d -= edge * np.round(d / edge)
            if np.min(np.einsum("ij,ij->i", d, d)) < oo_min * oo_min:
                continue
        q = rng.standard_normal(4)
        q /= np.linalg.norm(q)
        w, x, y, z = q
        R = np.array([
            [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
            [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
            [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])
        opos = np.vstack([opos, o])
        xyz.extend([o, o + R @ h1, o + R @ h2])
    return np.array(xyz)


def _psd_factor(rng, nao, nocc, scale):
    return rng.standard_normal((nao, nocc)) * scale


def _water_config(k, name, nmol, edge, meshes, o_ls, h_ls, nocc, deriv, seed):
    rng = np.random.default_rng(seed)
    o_exps = _loguniform(rng, 0.1, 12.0, len(o_ls))
    h_exps = _loguniform(rng, 0.1, 4.0, len(h_ls))
    xyz = _water_geometry(rng, nmol, edge)
    atom_shells = []
    for _ in range(nmol):
        atom_shells.append(_single_prim_shells(o_ls, o_exps))
        atom_shells.append(_single_prim_shells(h_ls, h_exps))
        atom_shells.append(_single_prim_shells(h_ls, h_exps))
    sa, sl, sn, so, pe, pc = pack_shells(atom_shells)
    nao = int(sum(ncart(int(l)) for l in sl))
    C = _psd_factor(rng, nao, nocc, 1.0 / math.sqrt(nao))
    return GPWInputs(name=name, cell=np.eye(3) * edge, xyz=xyz, shl_atom=sa, shl_l=sl,
                     shl_nprim=sn, shl_prim_off=so, prim_exp=pe, prim_coef=pc,
                     mesh=np.array([[m, m, m] for m in meshes], np.int32),
                     tau=1e-10, rel_cutoff=20.0, hermi=1, deriv=deriv, C=C, seed=seed)


def make_config(k: int, seed: Optional[int] = None) -> GPWInputs:
    """The k-th workload of BASELINE.json (k = 0..4)."""
    seed = BASE_SEED + k if seed is None else seed
    if k == 0:
        rng = np.random.default_rng(seed)
        o = np.array([5.0, 5.0, 5.0])
        xyz = np.array([o, o + [1.43, 1.11, 0.0], o + [-1.43, 1.11, 0.0]])
        o_ls, h_ls = [0, 0, 1, 1, 2], [0, 0, 1]
        atom_shells = [
            _single_prim_shells(o_ls, _loguniform(rng, 0.1, 10.0, 5)),
            _single_prim_shells(h_ls, _loguniform(rng, 0.1, 10.0, 3)),
            _single_prim_shells(h_ls, _loguniform(rng, 0.1, 10.0, 3)),
        ]
        sa, sl, sn, so, pe, pc = pack_shells(atom_shells)
        C = _psd_factor(rng, 24, 5, 0.3)
        return GPWInputs(name="cfg0_tiny", cell=np.eye(3) * 10.0, xyz=xyz, shl_atom=sa,
                         shl_l=sl, shl_nprim=sn, shl_prim_off=so, prim_exp=pe, prim_coef=pc,
                         mesh=np.array([[32, 32, 32]], np.int32), tau=1e-10,
                         rel_cutoff=20.0, hermi=1, deriv=0, C=C, seed=seed)
    if k == 1:
        return _water_config(1, "cfg1_32water_lda", 32, 18.6, [100, 60, 36, 20],
                             [0, 0, 1, 1, 2], [0, 0, 1], 128, 0, seed)
    if k == 2:
        return _water_config(2, "cfg2_256water_gga", 256, 37.2, [200, 120, 72, 40],
                             [0, 0, 1, 1, 2], [0, 0, 1], 1024, 1, seed)
    if k == 3:
        rng = np.random.default_rng(seed)
        a0, rep = 10.26, 2
        edge = a0 * rep
        cell = edge * (np.eye(3) + 0.08 * (np.ones((3, 3)) - np.eye(3)))
        basis = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]])
        basis = np.vstack([basis, basis + 0.25])
        frac = []
        for i in range(rep):
            for j in range(rep):
                for m in range(rep):
                    frac.extend((basis + [i, j, m]) / rep)
        frac = np.array(frac)
        xyz = frac @ cell
        ls = [0, 0, 1, 1, 2, 2, 3]
        exps = _loguniform(rng, 0.08, 6.0, 7)
        atom_shells = [_single_prim_shells(ls, exps) for _ in range(xyz.shape[0])]
        sa, sl, sn, so, pe, pc = pack_shells(atom_shells)
        nao = int(sum(ncart(int(l)) for l in sl))
        C = _psd_factor(rng, nao, 256, 1.0 / math.sqrt(nao))
        return GPWInputs(name="cfg3_diamond_f_triclinic", cell=cell, xyz=xyz, shl_atom=sa,
                         shl_l=sl, shl_nprim=sn, shl_prim_off=so, prim_exp=pe, prim_coef=pc,
                         mesh=np.array([[m, m, m] for m in (128, 80, 48, 28)], np.int32),
                         tau=1e-10, rel_cutoff=20.0, hermi=1, deriv=0, C=C, seed=seed)
    if k == 4:
        return _water_config(4, "cfg4_512water_gga_f", 512, 46.9, [256, 160, 96, 56, 32],
                             [0, 0, 1, 1, 2, 2, 3], [0, 0, 1], 2048, 1, seed)
    raise ValueError("config index must be 0..4")


def make_small(kind: str, seed: int = 1, deriv: int = 0, tau: float = 1e-10,
               hermi: int = 1) -> GPWInputs:
    """Small cells for tests: sized so that the dense plain-definition oracle
    (all lattice images) runs in seconds.

    kinds:
      'cubic'      2 atoms (s,p,d | s,p), cubic 7 Bohr, one 28^3 mesh
      'triclinic'  2 atoms (s,p,d,f | s,p,d), sheared cell, meshes 36x32x28 and 20x16x16
      'wrap'       1+1 atoms with diffuse shells in a 5 Bohr cell (R_t > cell edge), 16^3
      'ortho'      2 atoms, s..f / s..d, orthorhombic 6 x 7.5 x 9 Bohr, meshes 24x36x44, 12x20x24
      'contracted' 2 atoms, shells with 3 primitives each, cubic 8 Bohr, meshes 32^3, 16^3
      'resolved'   2 atoms, soft exponents on a fine mesh (a_p h^2 <= 0.3) for
                   quadrature-exact checks (v = 1 -> overlap; electron count)
    """
    rng = np.random.default_rng([BASE_SEED, 99, seed])
    rel = 20.0
    if kind == "cubic":
        cell = np.eye(3) * 7.0
        xyz = np.array([[1.3, 2.1, 3.2], [3.9, 4.4, 2.7]])
        shells = [_single_prim_shells([0, 1, 2], _loguniform(rng, 0.3, 3.0, 3)),
                  _single_prim_shells([0, 1], _loguniform(rng, 0.3, 3.0, 2))]
        mesh = [[28, 28, 28]]
    elif kind == "triclinic":
        cell = np.array([[6.5, 0.4, 0.3], [0.7, 6.0, -0.5], [-0.6, 0.9, 5.5]])
        xyz = np.array([[1.0, 1.5, 2.0], [3.3, 3.0, 2.6]])
        shells = [_single_prim_shells([0, 1, 2, 3], _loguniform(rng, 0.25, 2.5, 4)),
                  _single_prim_shells([0, 1, 2], _loguniform(rng, 0.25, 2.5, 3))]
        mesh = [[36, 32, 28], [20, 16, 16]]
    elif kind == "ortho":
        # orthorhombic, three different edges and meshes (ragged bricks along n2 and n3): the separable-Gaussian
        # path with a different metric, mesh and brick count per axis
        cell = np.diag([6.0, 7.5, 9.0])
        xyz = np.array([[1.1, 6.9, 2.0], [3.6, 3.0, 8.4]])
        shells = [_single_prim_shells([0, 1, 2, 3], _loguniform(rng, 0.25, 2.5, 4)),
                  _single_prim_shells([0, 1, 2], _loguniform(rng, 0.25, 2.5, 3))]
        mesh = [[24, 36, 44], [12, 20, 24]]
    elif kind == "wrap":
        cell = np.eye(3) * 5.0
        xyz = np.array([[0.7, 4.4, 2.5], [-0.9, 1.0, 6.1]])
        shells = [_single_prim_shells([0, 1], _loguniform(rng, 0.35, 1.2, 2)),
                  _single_prim_shells([0, 2], _loguniform(rng, 0.35, 1.2, 2))]
        mesh = [[16, 16, 16]]
    elif kind == "contracted":
        cell = np.eye(3) * 8.0
        xyz = np.array([[2.0, 2.5, 3.0], [4.6, 4.1, 3.7]])
        shells = []
        for ls in ([0, 1, 2], [0, 1]):
            sh = []
            for l in ls:
                exps = np.sort(_loguniform(rng, 0.3, 4.0, 3))[::-1]
                cs = rng.uniform(0.2, 1.0, 3)
                sh.append((l, list(exps), [float(c) * gto_norm(l, float(a)) for c, a in zip(cs, exps)]))
            shells.append(sh)
        mesh = [[32, 32, 32], [16, 16, 16]]
    elif kind == "resolved":
        cell = np.array([[8.0, 0.0, 0.0], [0.5, 7.5, 0.0], [0.2, -0.4, 7.0]])
        xyz = np.array([[2.0, 2.5, 3.0], [4.1, 4.3, 3.4]])
        shells = [_single_prim_shells([0, 1, 2, 3], _loguniform(rng, 0.25, 0.6, 4)),
                  _single_prim_shells([0, 1, 2], _loguniform(rng, 0.25, 0.6, 3))]
        mesh = [[48, 48, 44], [32, 32, 28]]
        rel = 100.0
    else:
        raise ValueError(kind)
    sa, sl, sn, so, pe, pc = pack_shells(shells)
    nao = int(sum(ncart(int(l)) for l in sl))
    C = _psd_factor(rng, nao, max(2, nao // 4), 0.4)
    return GPWInputs(name=f"small_{kind}", cell=np.asarray(cell, float), xyz=xyz, shl_atom=sa,
                     shl_l=sl, shl_nprim=sn, shl_prim_off=so, prim_exp=pe, prim_coef=pc,
                     mesh=np.array(mesh, np.int32), tau=tau, rel_cutoff=rel, hermi=hermi,
                     deriv=deriv, C=C, seed=int(BASE_SEED + 1000 + seed))


def make_custom(cell, xyz, atom_shells, mesh, C=None, tau=1e-10, rel_cutoff=20.0, hermi=1,
                deriv=0, seed=5, name="custom") -> GPWInputs:
    """Inputs from an explicit description: atom_shells[iatm] = [(l, [exps], [coefs]), ...]."""
    sa, sl, sn, so, pe, pc = pack_shells(atom_shells)
    nao = int(sum(ncart(int(l)) for l in sl))
    if C is None:
        rng = np.random.default_rng([BASE_SEED, 77, seed])
        C = _psd_factor(rng, nao, max(1, nao // 3), 0.5)
    return GPWInputs(name=name, cell=np.asarray(cell, float).reshape(3, 3),
                     xyz=np.asarray(xyz, float).reshape(-1, 3), shl_atom=sa, shl_l=sl,
                     shl_nprim=sn, shl_prim_off=so, prim_exp=pe, prim_coef=pc,
                     mesh=np.asarray(mesh, np.int32).reshape(-1, 3), tau=tau,
                     rel_cutoff=rel_cutoff, hermi=hermi, deriv=deriv,
                     C=np.asarray(C, float), seed=int(BASE_SEED + 2000 + seed))
