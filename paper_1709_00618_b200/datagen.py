"""Seeded synthetic TPC events (stand-ins for the ALICE data / Monte-Carlo the paper measures on).

This module is the ONE thing the CUDA path and the CPU oracle share: it produces *inputs* only
(cluster coordinates, the CSR row table and generator truth).  It holds none of the tracker's
arithmetic (no grid, no neighbour search, no Kalman filter, no selector).

Workloads follow BASELINE.json `configs[0..4]` (CFG:1-5) with the readings A14-A19 of
SURVEY.md §8(c); the recipe is restated in DESIGN.md §"Input recipe".

Conventions (SURVEY.md §8(c) "Geometry and units"): cm, Tesla, GeV/c.  Pad rows are planes
x = row_x[r] in the sector-local frame, x = X cos(a) + Y sin(a), y = -X sin(a) + Y cos(a),
z = Z, a = (s + 0.5) * 20 deg.  Sector instance s < 18 holds the z >= 0 side, s >= 18 the z < 0
side (side fixed by the un-shifted z).  Curvature kappa = c_B * q / pT, c_B = -0.00299792458 * Bz,
d(phi)/d(path) = kappa.

Random numbers: numpy Philox counter-based generator keyed by the integer seed, fp64 maths,
output rounded to fp32.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

N_ROWS = 159
X_FIRST = 85.0
X_LAST = 247.0
SECTORS_PER_SIDE = 18
SECTORS_PER_EVENT = 36
HALF_ANGLE_RAD = float(np.deg2rad(10.0))
Z_MAX = 250.0
C_LIGHT_KAPPA = 0.00299792458  # 1/cm per (T / (GeV/c))


def row_x(n_rows: int = N_ROWS) -> np.ndarray:
    """Pad-row radii, CFG:1: 159 rows at 85..247 cm spaced uniformly (fp32, as the tracker stores them)."""
    r = np.arange(n_rows, dtype=np.float64)
    return (X_FIRST + r * ((X_LAST - X_FIRST) / (n_rows - 1))).astype(np.float32)


def row_x_three_pad_sizes() -> np.ndarray:
    """159 pad rows with three pad lengths, as in the real TPC read-out chambers ("real TPC has 3
    pad sizes"): 63 rows of 0.75 cm, 64 rows of 1.0 cm, 32 rows of 1.5 cm, first row at 85 cm.  Used by the
    non-uniform-pitch reading A5'."""
    steps = np.concatenate([np.full(63, 0.75), np.full(64, 1.0), np.full(31, 1.5)])
    return (X_FIRST + np.concatenate([[0.0], np.cumsum(steps)])).astype(np.float32)


@dataclass
class Event:
    """One tracker input: `n_inst` sector instances, CSR over (instance, row)."""

    clusters: np.ndarray  # float32 [N,4] = (x, y, z, w); w carries the truth label as a float (-1 noise)
    row_offsets: np.ndarray  # int32 [n_inst*n_rows+1]
    labels: np.ndarray  # int32 [N] truth track id (unique within the event/window), -1 = noise
    n_inst: int
    n_rows: int
    bz: float
    z_lo: float
    z_hi: float
    sigma_y: float
    sigma_z: float
    truth: dict = field(default_factory=dict)  # per-track generator parameters (arrays indexed by label)
    name: str = ""
    rx: np.ndarray = None  # pad-row radii if they are not the uniform default (reading A5')

    @property
    def row_x(self) -> np.ndarray:
        return row_x(self.n_rows) if self.rx is None else self.rx

    @property
    def n_clusters(self) -> int:
        return int(self.clusters.shape[0])


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=int(seed)))


def _tracks(rng, n_prim, n_sec, *, single_sector, pt_mean=0.6, pt_min=0.1, eta_max=0.9, sec_radius=30.0):
    n = n_prim + n_sec
    pt = pt_min + rng.exponential(pt_mean - pt_min, n)  # A15
    eta = rng.uniform(-eta_max, eta_max, n)
    q = np.where(rng.uniform(size=n) < 0.5, -1.0, 1.0)
    if single_sector:  # A14: momentum azimuth inside sector 0's wedge, |eta| so that z >= 0
        phi0 = rng.uniform(0.0, 2.0 * HALF_ANGLE_RAD, n)
        eta = np.abs(eta)
    else:
        phi0 = rng.uniform(0.0, 2.0 * np.pi, n)
    org = np.zeros((n, 3))
    if n_sec:  # A17: uniform in a ball of radius 30 cm
        v = rng.normal(size=(n_sec, 3))
        v /= np.linalg.norm(v, axis=1)[:, None]
        rad = sec_radius * rng.uniform(size=n_sec) ** (1.0 / 3.0)
        org[n_prim:] = v * rad[:, None]
    return dict(pt=pt, eta=eta, q=q, phi0=phi0, x0=org[:, 0], y0=org[:, 1], z0=org[:, 2],
                primary=np.arange(n) < n_prim)


def _crossings(trk, bz, rx, sectors):
    """Pad-row plane intersections of each helix's first outgoing leg (A16). fp64.

    Returns arrays (sector 0..17, row, y, z, track index)."""
    rx = rx.astype(np.float64)
    tan_half = np.tan(HALF_ANGLE_RAD)
    kap = -C_LIGHT_KAPPA * bz * trk["q"] / trk["pt"]
    tl = np.sinh(trk["eta"])
    out = []
    for s in sectors:
        a = (s + 0.5) * 2.0 * HALF_ANGLE_RAD
        ca, sa = np.cos(a), np.sin(a)
        lx0 = trk["x0"] * ca + trk["y0"] * sa
        ly0 = -trk["x0"] * sa + trk["y0"] * ca
        pl = trk["phi0"] - a
        pl = (pl + np.pi) % (2.0 * np.pi) - np.pi
        sp, cp = np.sin(pl), np.cos(pl)
        # cheap pre-selection: only tracks that can reach this sector's +x half-space at all
        sel = np.nonzero(cp > -0.999)[0] if bz != 0.0 else np.nonzero(cp > 1e-3)[0]
        if sel.size == 0:
            continue
        dx = rx[None, :] - lx0[sel, None]
        if bz == 0.0:
            ok = dx > 0.0
            arc = dx / cp[sel, None]
            y = ly0[sel, None] + dx * (sp[sel] / cp[sel])[:, None]
            cpsi = np.broadcast_to(cp[sel, None], dx.shape)
            spsi = np.broadcast_to(sp[sel, None], dx.shape)
        else:
            k = kap[sel, None]
            sphi = sp[sel, None] + k * dx
            ok = np.abs(sphi) < 0.999
            sphi = np.clip(sphi, -0.999, 0.999)
            psi = np.arcsin(sphi)
            arc = (psi - pl[sel, None]) / k
            per = 2.0 * np.pi / np.abs(k)
            arc = np.where(arc < 0.0, arc + per, arc)
            ok &= (arc > 0.0) & (arc < 0.5 * per)
            cpsi = np.cos(psi)
            spsi = sphi
            y = ly0[sel, None] - (cpsi - cp[sel, None]) / k
        z = trk["z0"][sel, None] + arc * tl[sel, None]
        ok &= (np.abs(y) <= rx[None, :] * tan_half) & (np.abs(z) <= Z_MAX)
        ok &= (rx[None, :] * cpsi + y * spsi) > 0.0  # radially outward
        ti, ri = np.nonzero(ok)
        if ti.size:
            out.append((np.full(ti.size, s, np.int64), ri.astype(np.int64), y[ti, ri], z[ti, ri], sel[ti]))
    if not out:
        e = np.zeros(0)
        return e.astype(np.int64), e.astype(np.int64), e, e, e.astype(np.int64)
    return tuple(np.concatenate([o[i] for o in out]) for i in range(5))


def gen_clusters(rng, n_prim, n_sec, *, bz, eff, sigma_y, sigma_z, noise, single_sector, n_rows=N_ROWS, rx=None):
    """One collision: returns (inst, row, y, z, label) arrays + per-track truth. Noise label = -1."""
    rx = row_x(n_rows) if rx is None else rx
    trk = _tracks(rng, n_prim, n_sec, single_sector=single_sector)
    sectors = [0] if single_sector else range(SECTORS_PER_SIDE)
    sec, row, y, z, ti = _crossings(trk, bz, rx, sectors)
    inst = sec + SECTORS_PER_SIDE * (z < 0.0)
    if single_sector:
        keep = z >= 0.0
        inst, row, y, z, ti = inst[keep], row[keep], y[keep], z[keep], ti[keep]
    if eff < 1.0:
        keep = rng.uniform(size=inst.size) < eff
        inst, row, y, z, ti = inst[keep], row[keep], y[keep], z[keep], ti[keep]
    if sigma_y > 0.0:
        y = y + rng.normal(0.0, sigma_y, y.size)
    if sigma_z > 0.0:
        z = z + rng.normal(0.0, sigma_z, z.size)
    n_noise = int(round(noise * inst.size))  # A18
    if n_noise:
        ni = np.zeros(n_noise, np.int64) if single_sector else rng.integers(0, SECTORS_PER_EVENT, n_noise)
        nr = rng.integers(0, n_rows, n_noise)
        ny = rng.uniform(-1.0, 1.0, n_noise) * rx[nr].astype(np.float64) * np.tan(HALF_ANGLE_RAD)
        nz = rng.uniform(0.0, Z_MAX, n_noise) * np.where(ni >= SECTORS_PER_SIDE, -1.0, 1.0)
        inst = np.concatenate([inst, ni])
        row = np.concatenate([row, nr])
        y = np.concatenate([y, ny])
        z = np.concatenate([z, nz])
        ti = np.concatenate([ti, np.full(n_noise, -1, np.int64)])
    return inst, row, y, z, ti, trk


def _assemble(parts, truths, *, n_inst, n_rows, bz, z_lo, z_hi, sigma_y, sigma_z, name, inst_base=None, rx=None):
    """Merge per-collision cluster lists, sort per (instance,row) by (z,y) (A19), build the CSR table."""
    inst = np.concatenate([p[0] for p in parts])
    row = np.concatenate([p[1] for p in parts])
    y = np.concatenate([p[2] for p in parts]).astype(np.float32)
    z = np.concatenate([p[3] for p in parts]).astype(np.float32)
    lab = np.concatenate([p[4] for p in parts])
    key = inst * n_rows + row
    order = np.lexsort((y, z, key))
    key, y, z, lab = key[order], y[order], z[order], lab[order]
    counts = np.bincount(key, minlength=n_inst * n_rows)
    offs = np.zeros(n_inst * n_rows + 1, np.int64)
    np.cumsum(counts, out=offs[1:])
    rx_ = row_x(n_rows) if rx is None else rx
    cl = np.empty((y.size, 4), np.float32)
    cl[:, 0] = rx_[key % n_rows]
    cl[:, 1] = y
    cl[:, 2] = z
    cl[:, 3] = lab.astype(np.float32)
    truth = {k: np.concatenate([t[k] for t in truths]) for k in truths[0]} if truths else {}
    return Event(clusters=cl, row_offsets=offs.astype(np.int32), labels=lab.astype(np.int32), n_inst=n_inst,
                 n_rows=n_rows, bz=bz, z_lo=z_lo, z_hi=z_hi, sigma_y=sigma_y, sigma_z=sigma_z, truth=truth, name=name,
                 rx=rx)


def single_sector(seed=1001, n_tracks=200, *, bz=0.5, sigma_y=0.1, sigma_z=0.1, noise=0.02, eff=1.0,
                  n_rows=N_ROWS, rx=None) -> Event:
    """CFG:1 — one sector, 200 helices from the origin, smear 0.1 cm, 2 % noise (A14)."""
    rng = _rng(seed)
    inst, row, y, z, ti, trk = gen_clusters(rng, n_tracks, 0, bz=bz, eff=eff, sigma_y=sigma_y, sigma_z=sigma_z,
                                            noise=noise, single_sector=True, n_rows=n_rows, rx=rx)
    trk = dict(trk, z_shift=np.zeros(n_tracks))
    return _assemble([(inst, row, y, z, ti)], [trk], n_inst=1, n_rows=n_rows, bz=bz, z_lo=0.0, z_hi=Z_MAX,
                     sigma_y=max(sigma_y, 1e-3), sigma_z=max(sigma_z, 1e-3), name="cfg1_single_sector", rx=rx)


def full_event(seed=2001, n_prim=1000, *, sec_frac=0.0, bz=0.5, eff=0.95, sigma_y=0.1, sigma_z=0.1, noise=0.05,
               name="cfg2_peripheral", rx=None) -> Event:
    """CFG:2 (defaults) / CFG:3 (`central_event`) — 36 sectors, one collision."""
    rng = _rng(seed)
    n_sec = int(round(n_prim * sec_frac))
    inst, row, y, z, ti, trk = gen_clusters(rng, n_prim, n_sec, bz=bz, eff=eff, sigma_y=sigma_y, sigma_z=sigma_z,
                                            noise=noise, single_sector=False, rx=rx)
    trk = dict(trk, z_shift=np.zeros(n_prim + n_sec))
    return _assemble([(inst, row, y, z, ti)], [trk], n_inst=SECTORS_PER_EVENT, n_rows=N_ROWS, bz=bz, z_lo=0.0,
                     z_hi=Z_MAX, sigma_y=sigma_y, sigma_z=sigma_z, name=name, rx=rx)


def central_event(seed=3001, n_prim=8000) -> Event:
    """CFG:3 — 8,000 primaries + 20 % secondaries, smear 0.1 / 0.12 cm, 10 % noise, efficiency 0.95 (A17)."""
    return full_event(seed, n_prim, sec_frac=0.2, sigma_y=0.1, sigma_z=0.12, noise=0.10, name="cfg3_central")


def drift_window(seed=4001, n_events=5, *, mean_tracks=1500.0, cap_tracks=8000, bz=0.5, eff=0.95, sigma_y=0.1,
                 sigma_z=0.1, noise=0.10, max_shift=250.0) -> Event:
    """CFG:4 — `n_events` overlapping minimum-bias collisions, each shifted in z by U(-250,250) cm (A19)."""
    rng = _rng(seed)
    parts, truths = [], []
    base = 0
    for _ in range(n_events):
        n_trk = int(max(1, min(cap_tracks, rng.exponential(mean_tracks))))
        shift = float(rng.uniform(-max_shift, max_shift))
        inst, row, y, z, ti, trk = gen_clusters(rng, n_trk, 0, bz=bz, eff=eff, sigma_y=sigma_y, sigma_z=sigma_z,
                                                noise=noise, single_sector=False)
        z = z + shift  # side was fixed by the un-shifted z; no clipping
        parts.append((inst, row, y, z, np.where(ti >= 0, ti + base, -1)))
        truths.append(dict(trk, z_shift=np.full(n_trk, shift)))
        base += n_trk
    return _assemble(parts, truths, n_inst=SECTORS_PER_EVENT, n_rows=N_ROWS, bz=bz, z_lo=-max_shift,
                     z_hi=Z_MAX + max_shift, sigma_y=sigma_y, sigma_z=sigma_z, name="cfg4_drift_window")


def concat_events(events, name="batch") -> Event:
    """CFG:5 — a batch of independent windows = more sector instances (instance i has sector i % 36).

    Truth labels are offset so that they stay unique inside the batch."""
    e0 = events[0]
    cl = np.concatenate([e.clusters for e in events])
    labels, truths, base = [], [], 0
    offs = [np.zeros(1, np.int64)]
    cbase = 0
    for e in events:
        assert e.n_rows == e0.n_rows and e.bz == e0.bz and e.n_inst % SECTORS_PER_EVENT == 0 or len(events) == 1
        labels.append(np.where(e.labels >= 0, e.labels + base, -1))
        n_trk = len(e.truth["pt"]) if e.truth else 0
        base += n_trk
        truths.append(e.truth)
        offs.append(e.row_offsets[1:].astype(np.int64) + cbase)
        cbase += e.n_clusters
    lab = np.concatenate(labels).astype(np.int32)
    cl = cl.copy()
    cl[:, 3] = lab.astype(np.float32)
    truth = {k: np.concatenate([t[k] for t in truths]) for k in truths[0]} if truths[0] else {}
    return Event(clusters=cl, row_offsets=np.concatenate(offs).astype(np.int32), labels=lab,
                 n_inst=sum(e.n_inst for e in events), n_rows=e0.n_rows, bz=e0.bz,
                 z_lo=min(e.z_lo for e in events), z_hi=max(e.z_hi for e in events), sigma_y=e0.sigma_y,
                 sigma_z=e0.sigma_z, truth=truth, name=name, rx=e0.rx)


I16_Y_STEP = 1.0 / 256.0  # cm per count of the 16-bit fixed-point cluster format (include/tpc_tracker.h TPC_INPUT_I16)
I16_Z_STEP = 1.0 / 64.0


def quantise_i16(ev: Event):
    """The event in the 16-bit fixed-point input format: returns
    (q int16 [N,2], Event whose (y, z) are the decoded fp32 values).  Input formatting only: y = q_y / 256 cm (signed),
    z = z_origin + q_z / 64 cm (unsigned count), z_origin = z_lo on the z >= 0 side and -z_hi on the z < 0 side.
    The decoded event is what BOTH the oracle and the tracker see, so parity on quantised input stays exact."""
    inst = np.repeat(np.arange(ev.n_inst), np.diff(ev.row_offsets[::ev.n_rows]))
    z0 = np.where((inst % SECTORS_PER_EVENT) >= SECTORS_PER_SIDE, -ev.z_hi, ev.z_lo).astype(np.float32)
    y = ev.clusters[:, 1].astype(np.float64)
    z = ev.clusters[:, 2].astype(np.float64)
    qy = np.clip(np.rint(y / I16_Y_STEP), -32768, 32767).astype(np.int16)
    qz = np.clip(np.rint((z - z0.astype(np.float64)) / I16_Z_STEP), 0, 65535).astype(np.uint16)
    cl = ev.clusters.copy()
    cl[:, 1] = qy.astype(np.float32) * np.float32(I16_Y_STEP)               # exact
    cl[:, 2] = z0 + qz.astype(np.float32) * np.float32(I16_Z_STEP)          # exact product, one fp32 rounding
    q = np.stack([qy, qz.view(np.int16)], axis=1)
    from dataclasses import replace
    return np.ascontiguousarray(q), replace(ev, clusters=cl, name=ev.name + "_i16")


def window_batch(n_windows, seed0=5001, **kw) -> Event:
    """CFG:5 — `n_windows` CFG:4 drift windows, seeds seed0, seed0+1, ..."""
    return concat_events([drift_window(seed0 + w, **kw) for w in range(n_windows)], name=f"cfg5_batch{n_windows}")


def from_tracks(trk: dict, *, bz, sigma_y=0.0, sigma_z=0.0, eff=1.0, noise=0.0, seed=7, single=True,
                fp64_coords=False, rx=None):
    """Test helper: clusters of explicitly given tracks (dict with pt, eta, q, phi0, x0, y0, z0).

    Zero-smear / zero-noise / Bz=0 variants of CFG:1 used by the pins.  With
    `fp64_coords` the un-rounded fp64 (y, z) are returned next to the Event."""
    rng = _rng(seed)
    rx_arg = rx
    rx = row_x() if rx is None else rx
    trk = {k: np.asarray(v, dtype=np.float64) for k, v in trk.items()}
    sectors = [0] if single else range(SECTORS_PER_SIDE)
    sec, row, y, z, ti = _crossings(trk, bz, rx, sectors)
    inst = sec + SECTORS_PER_SIDE * (z < 0.0)
    if single:
        keep = z >= 0.0
        inst, row, y, z, ti = inst[keep], row[keep], y[keep], z[keep], ti[keep]
    if eff < 1.0:
        keep = rng.uniform(size=inst.size) < eff
        inst, row, y, z, ti = inst[keep], row[keep], y[keep], z[keep], ti[keep]
    if sigma_y > 0:
        y = y + rng.normal(0.0, sigma_y, y.size)
    if sigma_z > 0:
        z = z + rng.normal(0.0, sigma_z, z.size)
    n_noise = int(round(noise * inst.size))
    if n_noise:
        ni = np.zeros(n_noise, np.int64) if single else rng.integers(0, SECTORS_PER_EVENT, n_noise)
        nr = rng.integers(0, N_ROWS, n_noise)
        ny = rng.uniform(-1.0, 1.0, n_noise) * rx[nr].astype(np.float64) * np.tan(HALF_ANGLE_RAD)
        nz = rng.uniform(0.0, Z_MAX, n_noise) * np.where(ni >= SECTORS_PER_SIDE, -1.0, 1.0)
        inst, row = np.concatenate([inst, ni]), np.concatenate([row, nr])
        y, z, ti = np.concatenate([y, ny]), np.concatenate([z, nz]), np.concatenate([ti, np.full(n_noise, -1)])
    n_inst = 1 if single else SECTORS_PER_EVENT
    key = inst * N_ROWS + row
    order = np.lexsort((y.astype(np.float32), z.astype(np.float32), key))
    ev = _assemble([(inst, row, y, z, ti)], [dict(trk, z_shift=np.zeros(len(trk["pt"])),
                                                  primary=np.ones(len(trk["pt"]), bool))],
                   n_inst=n_inst, n_rows=N_ROWS, bz=bz, z_lo=0.0, z_hi=Z_MAX, sigma_y=max(sigma_y, 1e-3),
                   sigma_z=max(sigma_z, 1e-3), name="explicit_tracks", rx=rx_arg)
    if fp64_coords:
        return ev, y[order], z[order]
    return ev


def local_truth_state(trk: dict, idx: int, x: float, bz: float, sector: int = 0):
    """Generating helix of track `idx` expressed as the tracker's local state (y, z, sinPhi, dz/ds, q/pt)
    at sector-local plane `x` (first outgoing leg).  Used only by tests to compare fits with the truth."""
    a = (sector % SECTORS_PER_SIDE + 0.5) * 2.0 * HALF_ANGLE_RAD
    ca, sa = np.cos(a), np.sin(a)
    lx0 = trk["x0"][idx] * ca + trk["y0"][idx] * sa
    ly0 = -trk["x0"][idx] * sa + trk["y0"][idx] * ca
    pl = (trk["phi0"][idx] - a + np.pi) % (2.0 * np.pi) - np.pi
    k = -C_LIGHT_KAPPA * bz * trk["q"][idx] / trk["pt"][idx]
    tl = np.sinh(trk["eta"][idx])
    dx = x - lx0
    if bz == 0.0:
        return np.array([ly0 + dx * np.tan(pl), trk["z0"][idx] + dx / np.cos(pl) * tl, np.sin(pl), tl,
                         trk["q"][idx] / trk["pt"][idx]])
    sphi = np.sin(pl) + k * dx
    psi = np.arcsin(sphi)
    arc = (psi - pl) / k
    y = ly0 - (np.cos(psi) - np.cos(pl)) / k
    return np.array([y, trk["z0"][idx] + arc * tl + trk.get("z_shift", np.zeros(idx + 1))[idx], sphi, tl,
                     trk["q"][idx] / trk["pt"][idx]])
