"""Seeded synthetic plan generator (inputs only).

This module builds the *inputs* of the hot path -- the sparse spot->voxel influence
matrices D (dose) and L (LET-weighted dose), the voxel labels, the per-structure
bounds and the starting spot weights -- for the configurations that
BASELINE.json lists.  They stand in for the paper's two private patient plans
(sec. 2.1), which are not available; the structure follows the paper:
voxels x spots sparse matrices sharing one pattern, per-structure
bounds and weights, a PTV with adjacent OARs.

It holds NONE of the method's arithmetic (no projections, no residuals, no SpMV of
the iteration).  It serves both the CUDA path and the oracle; neither of them is
imported here.  All tensor work goes through torch so that the same code runs on
the CPU (tests) and on the GPU (large configs); values are evaluated in float64
and rounded ONCE to float32.

Geometry conventions:
  * voxel centre = (i + 1/2) h; linear voxel index x-fastest: ix + nx*(iy + ny*iz);
  * isocentre = grid centre;
  * a beam has a unit direction u and a flat entrance plane perpendicular to u at
    distance `d_iso` upstream of the isocentre (water phantom):
    depth(p) = (p - iso).u + d_iso;  r = distance from p to the spot axis;
  * spot index = beam-major, then energy layer, then lateral row-major.
Entries (BASELINE.json configs[0]):
  D_ij = Bragg(z; R_j) * exp(-r^2 / (2 sigma^2))      for r <= 3 sigma, 0 <= z <= R_j + 2 mm
  Bragg(z; R) = 0.3 + 0.7 exp(-(R - z)^2 / (2 * 2^2))  for z <= R,   exp(-(z - R)/1 mm) beyond
  LET(z; R)   = 2 + 10 exp(-max(R - z, 0) / 5 mm)      keV/um;       L_ij = LET * D_ij

Random numbers: a self-contained counter-based generator (splitmix64), not a
library default, so a seed means the same plan everywhere.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np
import torch

NAN = float("nan")
_M64 = (1 << 64) - 1


# --------------------------------------------------------------------------- RNG
def splitmix64(seed: int, counter: int) -> int:
    """One 64-bit output of splitmix64 at position `counter` of stream `seed`."""
    z = (seed * 0xD1342543DE82EF95 + (counter + 1) * 0x9E3779B97F4A7C15) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def uniform01(seed: int, counter: int) -> float:
    """Uniform double in [0, 1) from the top 53 bits."""
    return (splitmix64(seed, counter) >> 11) * (1.0 / (1 << 53))


def uniform01_array(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """Vectorised uniform01 for counters offset .. offset+n-1 (same values as the scalar form)."""
    with np.errstate(over="ignore"):
        c = np.arange(offset + 1, offset + n + 1, dtype=np.uint64)
        z = np.uint64((seed * 0xD1342543DE82EF95) & _M64) + c * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))


def log_uniform_weights(seed: int, n: int, lo_exp: float = -3.0) -> np.ndarray:
    """x = 10^(lo_exp * (1-U)), U uniform on [0,1): log-uniform over [1e-3, 1] (BASELINE.json configs[4])."""
    u = uniform01_array(seed, n)
    return np.power(10.0, lo_exp * (1.0 - u)).astype(np.float32)


# --------------------------------------------------------------------------- plan description
@dataclass
class Bounds:
    """Per-structure bounds; NaN = absent.  Mirrors `fredopt_bounds` in include/fredopt.h."""
    weight: float = 1.0
    dose_lo: float = NAN
    dose_hi: float = NAN
    dl_lo: float = NAN
    dl_hi: float = NAN
    letd_max: float = NAN
    dose_ref: float = NAN
    dl_ref: float = NAN

    def as_row(self) -> List[float]:
        return [self.weight, self.dose_lo, self.dose_hi, self.dl_lo, self.dl_hi,
                self.letd_max, self.dose_ref, self.dl_ref]


@dataclass
class Beam:
    u: Tuple[float, float, float]          # direction (normalised on use)
    d_iso: float                           # depth of the isocentre below the entrance plane [mm]
    pitch: float                           # lateral spot pitch [mm]
    n_layers: int
    sigma_lo: float                        # sigma at the deepest layer [mm]
    sigma_hi: float                        # sigma at the shallowest layer [mm]
    ranges: Optional[Sequence[float]] = None     # explicit ranges [mm]; default: across the PTV depth extent + 2 mm
    lattice: Optional[Tuple[int, int]] = None    # explicit (na, nb) lattice centred on the axis; default: PTV projection + 1 pitch


@dataclass
class Shape:
    """A structure: union of simple solids, optionally a shell around another label."""
    kind: str                              # "sphere" | "ellipsoid" | "cylinder" | "ring" | "bumpy"
    centre: Tuple[float, float, float] = (0.0, 0.0, 0.0)   # relative to the isocentre [mm]
    semi: Tuple[float, float, float] = (1.0, 1.0, 1.0)     # semi-axes; cylinder: (radius, radius, half-length)
    axis: int = 2                          # cylinder axis
    margin: float = 0.0                    # ring: thickness around label 1
    bump: Sequence[float] = ()             # bumpy: low-order surface perturbation coefficients


@dataclass
class PlanSpec:
    name: str
    grid: Tuple[int, int, int]
    h: float
    beams: List[Beam]
    structures: List[List[Shape]]          # structures[s-1] = solids whose union is label s; earlier labels win
    bounds: List[Bounds]
    n_iter: int
    lam: float = 1.0
    beta0: float = 1.0
    a: float = 0.99
    seed: int = 0
    label_all: bool = False                # configs[4]: every voxel labelled
    ptv_dose: float = 2.0


@dataclass
class Plan:
    spec: PlanSpec
    n_rows: int
    n_cols: int
    row_ptr: torch.Tensor                  # int64 [n_rows+1]
    col_idx: torch.Tensor                  # int32 [nnz], sorted within a row
    val_D: torch.Tensor                    # float32 [nnz]
    val_L: torch.Tensor                    # float32 [nnz]
    labels: torch.Tensor                   # int32 [n_rows]
    bounds: np.ndarray                     # float32 [n_struct, 8]
    x0: np.ndarray                         # float32 [n_cols]
    spot_range: np.ndarray = field(default=None)   # float64 [n_cols]  (for the analytic-LETd pin)
    spot_beam: np.ndarray = field(default=None)    # int32 [n_cols]

    @property
    def nnz(self) -> int:
        return int(self.col_idx.numel())

    def to_numpy(self):
        return (self.row_ptr.cpu().numpy(), self.col_idx.cpu().numpy(),
                self.val_D.cpu().numpy(), self.val_L.cpu().numpy(), self.labels.cpu().numpy())


# --------------------------------------------------------------------------- geometry helpers
def _unit(u):
    u = np.asarray(u, dtype=np.float64)
    return u / np.linalg.norm(u)


def _basis(u: np.ndarray):
    """Two unit vectors spanning the plane perpendicular to u (deterministic choice)."""
    k = int(np.argmin(np.abs(u)))
    t = np.zeros(3)
    t[k] = 1.0
    e1 = np.cross(u, t)
    e1 /= np.linalg.norm(e1)
    e2 = np.cross(u, e1)
    return e1, e2


def _voxel_centres(grid, h, device):
    nx, ny, nz = grid
    ix = (torch.arange(nx, device=device, dtype=torch.float64) + 0.5) * h
    iy = (torch.arange(ny, device=device, dtype=torch.float64) + 0.5) * h
    iz = (torch.arange(nz, device=device, dtype=torch.float64) + 0.5) * h
    # index order [iz, iy, ix] so that flattening gives the x-fastest linear index
    Z, Y, X = torch.meshgrid(iz, iy, ix, indexing="ij")
    return X, Y, Z


def _shape_mask(shape: Shape, X, Y, Z, iso, labels_so_far, h):
    cx, cy, cz = (iso[0] + shape.centre[0], iso[1] + shape.centre[1], iso[2] + shape.centre[2])
    dx, dy, dz = X - cx, Y - cy, Z - cz
    if shape.kind in ("sphere", "ellipsoid"):
        a, b, c = shape.semi
        return (dx / a) ** 2 + (dy / b) ** 2 + (dz / c) ** 2 <= 1.0
    if shape.kind == "cylinder":
        rad, _, half = shape.semi
        d = [dx, dy, dz]
        ax = shape.axis
        o = [i for i in range(3) if i != ax]
        return (d[o[0]] ** 2 + d[o[1]] ** 2 <= rad * rad) & (d[ax].abs() <= half)
    if shape.kind == "bumpy":
        a, b, c = shape.semi
        rho = torch.sqrt((dx / a) ** 2 + (dy / b) ** 2 + (dz / c) ** 2)
        rr = torch.sqrt(dx * dx + dy * dy + dz * dz).clamp_min(1e-9)
        nx_, ny_, nz_ = dx / rr, dy / rr, dz / rr
        bc = list(shape.bump) + [0.0] * 6
        pert = (bc[0] * nx_ + bc[1] * ny_ + bc[2] * nz_ + bc[3] * nx_ * ny_ + bc[4] * ny_ * nz_ + bc[5] * nz_ * nx_)
        return rho <= 1.0 + pert
    if shape.kind == "ring":
        # shell of thickness `margin` around label 1: dilate the PTV mask with a ball, via separable box passes
        # followed by an exact distance test on the (small) candidate set.
        ptv = labels_so_far == 1
        m = int(math.ceil(shape.margin / h))
        nzv, nyv, nxv = ptv.shape
        idx = ptv.nonzero()
        lo = (idx.min(0).values - m).clamp_min(0)
        hi = idx.max(0).values + m + 1
        hi = torch.minimum(hi, torch.tensor([nzv, nyv, nxv], device=hi.device))
        sub = ptv[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]].to(torch.float32)[None, None]
        k = torch.arange(-m, m + 1, device=sub.device, dtype=torch.float32) * h
        KZ, KY, KX = torch.meshgrid(k, k, k, indexing="ij")
        ball = ((KX * KX + KY * KY + KZ * KZ) <= shape.margin ** 2).to(torch.float32)[None, None]
        dil = torch.nn.functional.conv3d(sub, ball, padding=m)[0, 0] > 0.5
        out = torch.zeros_like(ptv)
        out[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]] = dil
        return out & ~ptv
    raise ValueError(shape.kind)


def build_labels(spec: PlanSpec, device) -> torch.Tensor:
    X, Y, Z = _voxel_centres(spec.grid, spec.h, device)
    iso = [spec.grid[0] * spec.h / 2.0, spec.grid[1] * spec.h / 2.0, spec.grid[2] * spec.h / 2.0]
    labels = torch.zeros(X.shape, dtype=torch.int32, device=device)
    for s, solids in enumerate(spec.structures, start=1):
        m = torch.zeros(X.shape, dtype=torch.bool, device=device)
        for sh in solids:
            m |= _shape_mask(sh, X, Y, Z, iso, labels, spec.h)
        labels = torch.where((labels == 0) & m, torch.full_like(labels, s), labels)   # earlier labels win (PTV first)
    if spec.label_all:
        labels = torch.where(labels == 0, torch.full_like(labels, len(spec.structures)), labels)
    return labels.reshape(-1)


# --------------------------------------------------------------------------- spots
def _beam_spots(spec: PlanSpec, beam: Beam, labels: torch.Tensor, device):
    """Returns per-spot arrays for one beam: lateral (a, b) [mm], range R [mm], sigma [mm]."""
    u = _unit(beam.u)
    e1, e2 = _basis(u)
    nx, ny, nz = spec.grid
    h = spec.h
    iso = np.array([nx * h / 2.0, ny * h / 2.0, nz * h / 2.0])
    ptv = (labels == 1).nonzero().reshape(-1)
    ix = ptv % nx
    iy = (ptv // nx) % ny
    iz = ptv // (nx * ny)
    P = torch.stack([(ix.double() + 0.5) * h - iso[0], (iy.double() + 0.5) * h - iso[1],
                     (iz.double() + 0.5) * h - iso[2]], dim=1)
    tu = torch.tensor(u, device=device)
    t1 = torch.tensor(e1, device=device)
    t2 = torch.tensor(e2, device=device)
    depth = P @ tu + beam.d_iso
    if beam.lattice is not None:
        na, nb = beam.lattice
        aa = (np.arange(na) - (na - 1) / 2.0) * beam.pitch
        bb = (np.arange(nb) - (nb - 1) / 2.0) * beam.pitch
        A, B = np.meshgrid(aa, bb, indexing="xy")          # row-major over b, a fastest
        lat_a, lat_b = A.reshape(-1), B.reshape(-1)
    else:
        ia = torch.round((P @ t1) / beam.pitch).long()
        ib = torch.round((P @ t2) / beam.pitch).long()
        a0, b0 = int(ia.min()) - 1, int(ib.min()) - 1
        na, nb = int(ia.max()) - a0 + 2, int(ib.max()) - b0 + 2
        occ = torch.zeros(nb, na, dtype=torch.float32, device=device)
        occ[ib - b0, ia - a0] = 1.0
        occ = torch.nn.functional.max_pool2d(occ[None, None], 3, stride=1, padding=1)[0, 0] > 0.5   # + one pitch
        jb, ja = occ.nonzero(as_tuple=True)                # row-major: b slow, a fast
        lat_a = ((ja + a0).double() * beam.pitch).cpu().numpy()
        lat_b = ((jb + b0).double() * beam.pitch).cpu().numpy()
    if beam.ranges is not None:
        ranges = np.asarray(beam.ranges, dtype=np.float64)
    else:
        zlo, zhi = float(depth.min()), float(depth.max()) + 2.0
        ranges = zlo + (zhi - zlo) * np.arange(beam.n_layers) / max(beam.n_layers - 1, 1)
    nl = len(ranges)
    if nl > 1:
        sig = beam.sigma_hi + (beam.sigma_lo - beam.sigma_hi) * np.arange(nl) / (nl - 1)   # shallow = broad
    else:
        sig = np.array([beam.sigma_lo])
    n_lat = len(lat_a)
    A = np.tile(lat_a, nl)
    B = np.tile(lat_b, nl)
    R = np.repeat(ranges, n_lat)
    S = np.repeat(sig, n_lat)
    return u, e1, e2, A, B, R, S


def _spot_entries(spec: PlanSpec, beam: Beam, u, e1, e2, A, B, R, S, col0: int, device, max_cand: int):
    """COO entries (row, col, D, L) of the spots of one beam, spot-major, batched over spots."""
    nx, ny, nz = spec.grid
    h = spec.h
    dims = [nx, ny, nz]
    iso = np.array([nx * h / 2.0, ny * h / 2.0, nz * h / 2.0])
    ax = int(np.argmax(np.abs(u)))
    o1, o2 = [i for i in range(3) if i != ax]
    K = dims[ax]
    rows_out, cols_out, d_out, l_out = [], [], [], []
    n_spots = len(A)
    kk = (torch.arange(K, device=device, dtype=torch.float64) + 0.5) * h          # slice coordinates along ax
    j = 0
    while j < n_spots:
        sig_max = float(S[j])
        m = int(math.ceil(3.0 * sig_max / (h * abs(u[ax])))) + 1
        w = 2 * m + 1
        nb = max(1, min(n_spots - j, max_cand // (K * w * w)))
        # keep a batch within one sigma value (sigma is constant within a layer) so that m is shared
        same = np.nonzero(S[j:j + nb] != S[j])[0]
        if same.size:
            nb = int(same[0])
        sl = slice(j, j + nb)
        p0 = (iso[None, :] + A[sl, None] * e1[None, :] + B[sl, None] * e2[None, :])           # [nb, 3] axis point at the iso plane
        p0 = torch.tensor(p0, device=device)
        tu = torch.tensor(u, device=device)
        Rj = torch.tensor(R[sl], device=device)[:, None, None]
        Sj = torch.tensor(S[sl], device=device)[:, None, None]
        t = (kk[None, :] - p0[:, ax:ax + 1]) / u[ax]                                          # [nb, K]
        c1 = p0[:, o1:o1 + 1] + t * u[o1]
        c2 = p0[:, o2:o2 + 1] + t * u[o2]
        i1c = torch.floor(c1 / h).long()
        i2c = torch.floor(c2 / h).long()
        off = torch.arange(-m, m + 1, device=device)
        O1 = off.repeat_interleave(w)[None, None, :]                                          # [1,1,w*w]
        O2 = off.repeat(w)[None, None, :]
        i1 = i1c[:, :, None] + O1
        i2 = i2c[:, :, None] + O2
        q1 = (i1.double() + 0.5) * h
        q2 = (i2.double() + 0.5) * h
        qa = kk[None, :, None]
        w1 = q1 - p0[:, o1, None, None]
        w2 = q2 - p0[:, o2, None, None]
        wa = qa - p0[:, ax, None, None]
        along = w1 * u[o1] + w2 * u[o2] + wa * u[ax]
        r2 = (w1 * w1 + w2 * w2 + wa * wa - along * along).clamp_min(0.0)
        z = along + beam.d_iso
        keep = (r2 <= 9.0 * Sj * Sj) & (z <= Rj + 2.0) & (z >= 0.0)
        keep &= (i1 >= 0) & (i1 < dims[o1]) & (i2 >= 0) & (i2 < dims[o2])
        sel = keep.nonzero(as_tuple=True)
        zs, r2s = z[sel], r2[sel]
        Rs = Rj.expand_as(z)[sel]
        Ss = Sj.expand_as(z)[sel]
        prox = Rs - zs
        bragg = torch.where(prox >= 0.0, 0.3 + 0.7 * torch.exp(-(prox * prox) / 8.0), torch.exp(prox / 1.0))
        dval = bragg * torch.exp(-r2s / (2.0 * Ss * Ss))
        let = 2.0 + 10.0 * torch.exp(-prox.clamp_min(0.0) / 5.0)
        lval = let * dval
        idx = [None, None, None]
        idx[ax] = sel[1]
        idx[o1] = i1[sel]
        idx[o2] = i2[sel]
        row = idx[0] + nx * (idx[1] + ny * idx[2])
        col = sel[0] + (col0 + j)
        d32 = dval.float()
        l32 = lval.float()
        nzmask = d32 > 0                                   # underflow to 0 in fp32 cannot occur here, but keep the pattern honest
        rows_out.append(row[nzmask].int())
        cols_out.append(col[nzmask].int())
        d_out.append(d32[nzmask])
        l_out.append(l32[nzmask])
        j += nb
    return rows_out, cols_out, d_out, l_out


def build_plan(spec: PlanSpec, device: str = "cpu", max_cand: int = 1 << 24) -> Plan:
    """Generate the plan `spec` on `device`.  Tensors stay on that device."""
    dev = torch.device(device)
    labels = build_labels(spec, dev)
    nx, ny, nz = spec.grid
    V = nx * ny * nz
    rows_l, cols_l, d_l, l_l = [], [], [], []
    col0 = 0
    spot_range, spot_beam = [], []
    for b, beam in enumerate(spec.beams):
        u, e1, e2, A, B, R, S = _beam_spots(spec, beam, labels, dev)
        r_, c_, dv_, lv_ = _spot_entries(spec, beam, u, e1, e2, A, B, R, S, col0, dev, max_cand)
        rows_l += r_
        cols_l += c_
        d_l += dv_
        l_l += lv_
        col0 += len(A)
        spot_range.append(R)
        spot_beam.append(np.full(len(A), b, dtype=np.int32))
    S_tot = col0
    rows = torch.cat(rows_l)
    del rows_l
    cols = torch.cat(cols_l)
    del cols_l
    vd = torch.cat(d_l)
    del d_l
    vl = torch.cat(l_l)
    del l_l
    # CSR: stable sort by row keeps the spot-major generation order inside a row => columns ascending
    rows_sorted, perm = torch.sort(rows, stable=True)
    del rows
    cols = cols[perm]
    vd = vd[perm]
    vl = vl[perm]
    del perm
    counts = torch.bincount(rows_sorted.long(), minlength=V)
    row_ptr = torch.zeros(V + 1, dtype=torch.int64, device=dev)
    torch.cumsum(counts, 0, out=row_ptr[1:])
    # starting weights: uniform, mean PTV dose = ptv_dose; computed once in fp64, rounded to fp32
    ptv_rows = labels[rows_sorted.long()] == 1
    tot = vd[ptv_rows].double().sum().item()
    n_ptv = int((labels == 1).sum().item())
    x0v = spec.ptv_dose * n_ptv / tot if tot > 0 else 1.0
    x0 = np.full(S_tot, x0v, dtype=np.float64).astype(np.float32)
    del rows_sorted
    bounds = np.array([b.as_row() for b in spec.bounds], dtype=np.float32)
    return Plan(spec=spec, n_rows=V, n_cols=S_tot, row_ptr=row_ptr, col_idx=cols, val_D=vd, val_L=vl,
                labels=labels, bounds=bounds, x0=x0,
                spot_range=np.concatenate(spot_range), spot_beam=np.concatenate(spot_beam))


# --------------------------------------------------------------------------- the configurations of BASELINE.json
def config_spec(i: int, seed: int = 0, scale: float = 1.0) -> PlanSpec:
    """PlanSpec for BASELINE.json configs[i] (i = 0..3).  configs[4] (the pass sweep) is `sweep_spec`."""
    if i == 0:
        # Tiny phantom: 32^3 @ 3 mm, one beam +z, 10x10 spots @ 3 mm x 8 layers (ranges 40..70 mm), sigma 4 mm
        return PlanSpec(
            name="config0_tiny", grid=(32, 32, 32), h=3.0,
            beams=[Beam(u=(0, 0, 1), d_iso=48.0, pitch=3.0, n_layers=8, sigma_lo=4.0, sigma_hi=4.0,
                        ranges=[40.0 + e * 30.0 / 7.0 for e in range(8)], lattice=(10, 10))],
            structures=[[Shape("sphere", (0, 0, 0), (15, 15, 15))],
                        [Shape("ellipsoid", (0, 0, 23), (15, 15, 8))]],
            bounds=[Bounds(1.0, dose_lo=0.95 * 2, dose_hi=1.07 * 2, dose_ref=2.0),
                    Bounds(1.0, dose_hi=1.5, letd_max=4.0)],
            n_iter=50, lam=1.0, beta0=1.0, a=0.99, seed=seed)
    if i == 1:
        # Mid-size single field: 96^3 @ 2 mm, 5 mm pitch over the PTV projection, 25 layers, sigma 5 mm
        return PlanSpec(
            name="config1_mid", grid=(96, 96, 96), h=2.0,
            beams=[Beam(u=(0, 0, 1), d_iso=96.0, pitch=5.0, n_layers=25, sigma_lo=5.0, sigma_hi=5.0)],
            structures=[[Shape("sphere", (0, 0, 0), (30, 30, 30))],
                        [Shape("ellipsoid", (0, 0, 42), (28, 28, 12))],
                        [Shape("cylinder", (44, 0, 0), (13, 13, 30), axis=1)]],
            bounds=[Bounds(1.0, dose_lo=0.95 * 2, dose_hi=1.07 * 2, dose_ref=2.0),
                    Bounds(1.0, dose_hi=1.5, dl_hi=6.0, letd_max=4.0, dl_ref=6.0),
                    Bounds(1.0, dose_hi=1.5, dl_hi=6.0, letd_max=4.0, dl_ref=6.0)],
            n_iter=200, seed=seed)
    if i == 2:
        # Brain-tumour-shaped: 256x256x160 @ 2 mm, coplanar beams 0/90/270 deg, 4 mm pitch, sigma 3..7 mm
        c = [(uniform01(seed, 10 + 3 * k) - 0.5, uniform01(seed, 11 + 3 * k) - 0.5, uniform01(seed, 12 + 3 * k) - 0.5)
             for k in range(3)]
        rad = [17.0 + 3.0 * uniform01(seed, 30 + k) for k in range(3)]
        ptv = [Shape("sphere", (24.0 * c[k][0], 24.0 * c[k][1], 16.0 * c[k][2]), (rad[k],) * 3) for k in range(3)]
        g = (int(256 * scale), int(256 * scale), int(160 * scale))
        return PlanSpec(
            name="config2_brain", grid=g, h=2.0,
            beams=[Beam(u=(0, 1, 0), d_iso=110.0, pitch=4.0, n_layers=25, sigma_lo=3.0, sigma_hi=7.0),
                   Beam(u=(1, 0, 0), d_iso=100.0, pitch=4.0, n_layers=25, sigma_lo=3.0, sigma_hi=7.0),
                   Beam(u=(-1, 0, 0), d_iso=100.0, pitch=4.0, n_layers=25, sigma_lo=3.0, sigma_hi=7.0)],
            structures=[ptv,
                        [Shape("cylinder", (0, -40, 0), (10, 10, 24), axis=2)],      # brainstem-like
                        [Shape("ellipsoid", (0, 34, 6), (9, 4, 3))],                 # chiasm-like
                        [Shape("ring", margin=10.0)]],                              # normal-tissue ring
            bounds=[Bounds(1.0, dose_lo=0.95 * 2, dose_hi=1.07 * 2, dose_ref=2.0),
                    Bounds(1.0, dose_hi=1.5, dl_hi=6.0, letd_max=4.0, dl_ref=6.0),
                    Bounds(1.0, dose_hi=1.5, dl_hi=6.0, letd_max=4.0, dl_ref=6.0),
                    Bounds(1.0, dose_hi=2.14, dl_hi=8.0, dl_ref=8.0)],
            n_iter=500, seed=seed)
    if i == 3:
        # Large target: 300x300x200 @ 2 mm, three non-coplanar beams, ~30k spots, PTV ~600 cm^3 bumpy ellipsoid
        bump = [0.10 * (uniform01(seed, 50 + k) - 0.5) for k in range(6)]
        g = (int(300 * scale), int(300 * scale), int(200 * scale))
        return PlanSpec(
            name="config3_large", grid=g, h=2.0,
            beams=[Beam(u=(0.0, 1.0, 0.25), d_iso=200.0, pitch=5.0, n_layers=22, sigma_lo=5.5, sigma_hi=9.5),
                   Beam(u=(0.9, 0.3, -0.3), d_iso=200.0, pitch=5.0, n_layers=22, sigma_lo=5.5, sigma_hi=9.5),
                   Beam(u=(-0.85, 0.35, 0.4), d_iso=200.0, pitch=5.0, n_layers=22, sigma_lo=5.5, sigma_hi=9.5)],
            structures=[[Shape("bumpy", (0, 0, 0), (60, 55, 43), bump=bump)],
                        [Shape("cylinder", (0, -72, 0), (12, 12, 40), axis=2)],
                        [Shape("ellipsoid", (78, 0, 0), (14, 20, 16))],
                        [Shape("ellipsoid", (-80, 6, 0), (16, 18, 20))],
                        [Shape("ellipsoid", (0, 10, 62), (25, 25, 14))],
                        [Shape("ellipsoid", (10, 70, -10), (20, 11, 18))]],
            bounds=[Bounds(1.0, dose_lo=0.95 * 2, dose_hi=1.07 * 2, dose_ref=2.0),
                    Bounds(1.0, dose_hi=1.5, dl_hi=6.0, letd_max=4.0, dl_ref=6.0),
                    Bounds(1.0, dose_hi=1.5, dl_hi=6.0, letd_max=4.0, dl_ref=6.0),
                    Bounds(1.0, dose_hi=1.5, dl_hi=6.0, letd_max=4.0, dl_ref=6.0),
                    Bounds(1.0, dose_hi=1.6, dl_hi=7.0, dl_ref=7.0),
                    Bounds(1.0, dose_hi=1.5, dl_hi=6.0, letd_max=5.0, dl_ref=6.0)],
            n_iter=500, seed=seed)
    raise ValueError("config index must be 0..3 (configs[4] is the pass sweep: sweep_spec)")


def sweep_spec(sigma: float, pitch: float, n_layers: int, seed: int = 0, scale: float = 1.0) -> PlanSpec:
    """configs[4]: config-2 geometry, every voxel labelled, sigma and nnz (via pitch/layers) swept."""
    sp = config_spec(2, seed=seed, scale=scale)
    sp.name = f"sweep_sigma{sigma:g}_pitch{pitch:g}_layers{n_layers}"
    for b in sp.beams:
        b.sigma_lo = b.sigma_hi = sigma
        b.pitch = pitch
        b.n_layers = n_layers
    sp.label_all = True
    return sp


def random_small_plan(seed: int, V: int = 40, S: int = 8, n_struct: int = 3, density: float = 0.4,
                      same_pattern: bool = True):
    """Tiny random CSR problem for brute-force checks (numpy arrays).  Not plan-shaped on purpose."""
    u = uniform01_array(seed, 4 * V * S + V + S + 64)
    k = 0
    mask = (u[k:k + V * S] < density).reshape(V, S); k += V * S
    Dd = (0.05 + u[k:k + V * S]).reshape(V, S) * mask; k += V * S
    let = 2.0 + 8.0 * u[k:k + V * S].reshape(V, S); k += V * S
    Ld = Dd * let
    # different patterns: L's mask is drawn INDEPENDENTLY of D's, so rows hold entries in D only, in L only and in both
    maskL = mask if same_pattern else (u[k:k + V * S] < density).reshape(V, S)
    k += V * S
    if not same_pattern:
        Ld = np.where(maskL, np.where(mask, Ld, 0.3 * let), 0.0)
    labels = np.floor(u[k:k + V] * (n_struct + 1)).astype(np.int32); k += V
    labels = np.minimum(labels, n_struct)

    def csr(M, msk):
        rp = np.zeros(V + 1, dtype=np.int64)
        ci, vv = [], []
        for i in range(V):
            js = np.nonzero(msk[i])[0]
            rp[i + 1] = rp[i] + len(js)
            ci.append(js.astype(np.int32))
            vv.append(M[i, js].astype(np.float32))
        return rp, (np.concatenate(ci) if ci else np.zeros(0, np.int32)), \
            (np.concatenate(vv) if vv else np.zeros(0, np.float32))

    D = csr(Dd, mask)
    L = csr(Ld, maskL)
    x0 = (0.2 + u[k:k + S]).astype(np.float32)
    return D, L, labels, x0
