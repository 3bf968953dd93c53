"""Seeded, synthetic input generators shared by the oracle harness and the CUDA path.

This module holds NONE of the method's arithmetic: it only builds the *inputs*
(phantom volumes, material compositions, beam descriptions, run sizes) of the
five BASELINE.json configs plus a few tiny test cases.  Both `oracle/` and the
CUDA library receive exactly these numpy arrays / plain dicts.

Workload shapes follow PAPER.md:82-86 (§2.2 Materials: water / slab / half-slab
phantoms, point source at SSD 100 cm, 15 MeV electrons and a 6 MV photon
spectrum) as re-stated by BASELINE.json `configs` (10x10 cm^2 fields, 0.5 /
0.25 cm voxels).  The 6 MV spectrum is not printed in the paper; the synthetic
triangular spectrum of BASELINE.json config 3 stands in for it.
"""
from __future__ import annotations

import numpy as np

# --- materials (user input per PAPER.md:31 "user-defined material composition") ---------------
# (Z, A, mass fraction) triples; I in eV; nominal density in g/cm^3.  Compositions are the
# harness's choice (the paper prints none); both sides get the same numbers.
_A = {1: 1.008, 6: 12.011, 7: 14.007, 8: 15.999, 11: 22.990, 12: 24.305, 15: 30.974,
      16: 32.06, 17: 35.45, 19: 39.098, 20: 40.078}


def _mat(name, fractions, I_eV, rho):
    Z = np.array(sorted(fractions), dtype=np.int32)
    w = np.array([fractions[z] for z in Z], dtype=np.float64)
    w = w / w.sum()
    A = np.array([_A[int(z)] for z in Z], dtype=np.float64)
    return {"name": name, "Z": Z, "A": A.astype(np.float32), "w": w.astype(np.float32),
            "I_eV": float(I_eV), "rho_nominal": float(rho)}


def water():
    return _mat("water", {1: 0.1119, 8: 0.8881}, 75.0, 1.00)


def bone():
    return _mat("bone", {1: .064, 6: .278, 7: .027, 8: .410, 12: .002, 15: .070, 16: .002, 20: .147},
                91.9, 1.85)


def lung():
    return _mat("lung", {1: .103, 6: .105, 7: .031, 8: .749, 11: .002, 15: .002, 16: .003, 17: .003,
                         19: .002}, 75.3, 0.26)


MATERIALS = (water, bone, lung)  # material index 0, 1, 2


def materials(n=3):
    return [f() for f in MATERIALS[:n]]


# --- run parameters (cut-offs per BASELINE.json configs; step limits per DESIGN.md R2) ---------
def params(e_cut=0.2, g_cut=0.01, e_max=20.0, n_grid=256, d_maxs=0.5, f_maxe=0.2, flags=0):
    return {"e_cut_MeV": e_cut, "g_cut_MeV": g_cut, "e_max_MeV": e_max, "n_grid": n_grid,
            "d_maxs_cm": d_maxs, "f_maxe": f_maxe, "flags": flags}


FLAG_NO_HARD = 1        # no Moller / bremsstrahlung events
FLAG_NO_MS = 2          # no multiple-scattering deflection
FLAG_LOCAL_SECONDARIES = 4  # secondaries are deposited where they are born
FLAG_MS_GS = 8          # Goudsmit-Saunderson multiple-scattering angle instead of the Gaussian model (R27)
FLAG_MULTI_VOXEL = 16   # electron steps are not limited by the voxel: they cross faces (gDPM-style stepping; R28)


# --- phantoms ------------------------------------------------------------------------------------
def _phantom(dims, voxel, origin, mat, rho):
    return {"dims": np.array(dims, dtype=np.int32), "voxel_cm": np.array(voxel, dtype=np.float32),
            "origin_cm": np.array(origin, dtype=np.float32),
            "material": np.ascontiguousarray(mat, dtype=np.uint8).reshape(-1),
            "density": np.ascontiguousarray(rho, dtype=np.float32).reshape(-1)}


def homogeneous_phantom(dims, voxel_cm, origin=None, material=0, density=1.0):
    nx, ny, nz = dims
    h = (voxel_cm,) * 3 if np.isscalar(voxel_cm) else tuple(voxel_cm)
    if origin is None:
        origin = (-0.5 * nx * h[0], -0.5 * ny * h[1], 0.0)
    n = nx * ny * nz
    return _phantom(dims, h, origin, np.full(n, material, np.uint8), np.full(n, density, np.float32))


def slab_phantom(dims=(61, 61, 60), voxel_cm=0.5, half=False):
    """water 0-3 cm, bone 3-5 cm (1.85), lung 5-12 cm (0.26), water 12-30 cm (BASELINE configs 4, 5).
    Array layout: x fastest, i = ix + nx*(iy + ny*iz).  half=True: heterogeneity only for ix < nx/2."""
    nx, ny, nz = dims
    h = float(voxel_cm)
    mat = np.zeros((nz, ny, nx), np.uint8)
    rho = np.ones((nz, ny, nx), np.float32)
    zc = (np.arange(nz) + 0.5) * h
    xs = slice(0, nx // 2) if half else slice(0, nx)
    for iz in range(nz):
        if 3.0 < zc[iz] < 5.0:
            mat[iz, :, xs] = 1
            rho[iz, :, xs] = 1.85
        elif 5.0 < zc[iz] < 12.0:
            mat[iz, :, xs] = 2
            rho[iz, :, xs] = 0.26
    return _phantom(dims, (h, h, h), (-0.5 * nx * h, -0.5 * ny * h, 0.0), mat, rho)


# --- beams ---------------------------------------------------------------------------------------
PHOTON, ELECTRON, POSITRON = 0, -1, 1
PENCIL, POINT_RECT = 0, 1


def beam(particle, shape, energy=None, spectrum=None, field=(10.0, 10.0), ssd=100.0,
         entry=(0.0, 0.0, 0.0)):
    if spectrum is None:
        E = np.array([energy], np.float32)
        p = np.array([1.0], np.float32)
    else:
        E, p = (np.asarray(a, np.float32) for a in spectrum)
    return {"particle": int(particle), "shape": int(shape), "entry_cm": np.array(entry, np.float32),
            "axis": np.array((0, 0, 1), np.float32), "ssd_cm": float(ssd),
            "field_cm": np.array(field, np.float32), "E_nodes_MeV": E, "pdf_nodes": p}


def spectrum_6mv():
    """BASELINE.json config 3: piecewise-linear pdf on 0.25..6 MeV in 0.25 MeV bins, 0 at 0.25,
    peak at 1.0, falling linearly to 0 at 6.0 (24 nodes)."""
    E = np.arange(1, 25, dtype=np.float64) * 0.25
    p = np.where(E <= 1.0, (E - 0.25) / 0.75, (6.0 - E) / 5.0)
    return E.astype(np.float32), p.astype(np.float32)


def electron_pencil(E=6.0):
    return beam(ELECTRON, PENCIL, energy=E)


def electron_field(E=15.0):
    return beam(ELECTRON, POINT_RECT, energy=E)


def photon_field():
    return beam(PHOTON, POINT_RECT, spectrum=spectrum_6mv())


def paper_slab_phantom(half=False):
    """The paper's phantoms: 32 cm cube at 0.25 cm voxels (128^3); slab = water 0-2 cm, bone 2-4 cm,
    lung 4-6 cm, water below; half-slab = the bone and lung layers cover half of the xoy plane (x < 0)."""
    n, h = 128, 0.25
    mat = np.zeros((n, n, n), np.uint8)
    rho = np.ones((n, n, n), np.float32)
    zc = (np.arange(n) + 0.5) * h
    xs = slice(0, n // 2) if half else slice(0, n)
    for iz in range(n):
        if 2.0 < zc[iz] < 4.0:
            mat[iz, :, xs] = 1
            rho[iz, :, xs] = 1.85
        elif 4.0 < zc[iz] < 6.0:
            mat[iz, :, xs] = 2
            rho[iz, :, xs] = 0.26
    return _phantom((n, n, n), (h, h, h), (-0.5 * n * h, -0.5 * n * h, 0.0), mat, rho)


def paper_config(idx):
    """The five cases of the paper's Tables 2 and 3 with this build's physics: 128^3 x 0.25 cm
    phantoms, 2x2 cm^2 field at SSD 100 cm, 15 MeV electrons (5e6 histories) or the synthetic 6 MV spectrum (5e8),
    absorption energies 200 keV (electrons) / 50 keV (photons).  Context beside the paper's timings, not a target.
    idx: 1 e- water, 2 e- slab, 3 photon water, 4 photon slab, 5 photon half-slab."""
    names = {1: "p1_15MeV_e_water128", 2: "p2_15MeV_e_slab128", 3: "p3_6MV_g_water128", 4: "p4_6MV_g_slab128",
             5: "p5_6MV_g_halfslab128"}
    if idx not in names:
        raise ValueError("paper config index 1..5")
    if idx in (1, 3):
        ph = homogeneous_phantom((128, 128, 128), 0.25)
    else:
        ph = paper_slab_phantom(half=(idx == 5))
    if idx <= 2:
        bm, n = beam(ELECTRON, POINT_RECT, energy=15.0, field=(2.0, 2.0)), 5 * 10**6
    else:
        bm, n = beam(PHOTON, POINT_RECT, spectrum=spectrum_6mv(), field=(2.0, 2.0)), 5 * 10**8
    return {"phantom": ph, "materials": materials(3), "params": params(e_cut=0.2, g_cut=0.05), "beam": bm,
            "n_histories": n, "seed": 1, "n_batches": 10, "name": names[idx]}


# --- the five BASELINE.json configs -------------------------------------------------------------
def config(idx, beam_kind=None):
    """Return dict(phantom, materials, params, beam, n_histories, seed, n_batches, name).
    idx 1..5 as in BASELINE.json `configs` (1-based); configs 4 and 5 take beam_kind 'e' or 'g'.
    idx 'p1'..'p5': the paper-shaped cases of paper_config()."""
    if isinstance(idx, str) and idx.startswith("p"):
        return paper_config(int(idx[1:]))
    idx = int(idx)
    if idx == 1:
        ph, bm, n, B, name = homogeneous_phantom((20, 20, 20), 0.5), electron_pencil(6.0), 10**5, 10, \
            "c1_6MeV_e_pencil_water20"
    elif idx == 2:
        ph, bm, n, B, name = homogeneous_phantom((61, 61, 60), 0.5), electron_field(15.0), 10**7, 10, \
            "c2_15MeV_e_water61"
    elif idx == 3:
        ph, bm, n, B, name = homogeneous_phantom((61, 61, 60), 0.5), photon_field(), 10**8, 10, \
            "c3_6MV_g_water61"
    elif idx == 4:
        ph = slab_phantom()
        if beam_kind == "g":
            bm, n, name = photon_field(), 10**8, "c4_6MV_g_slab61"
        else:
            bm, n, name = electron_field(15.0), 10**7, "c4_15MeV_e_slab61"
        B = 10
    elif idx == 5:
        ph = slab_phantom((122, 122, 120), 0.25, half=True)
        if beam_kind == "e":
            bm, n, name = electron_field(15.0), 10**8, "c5_15MeV_e_halfslab122"
        else:
            bm, n, name = photon_field(), 10**9, "c5_6MV_g_halfslab122"
        B = 20
    else:
        raise ValueError("config index 1..5")
    return {"phantom": ph, "materials": materials(3), "params": params(), "beam": bm,
            "n_histories": n, "seed": 1, "n_batches": B, "name": name}


# --- particle-list ("phase-space") source ---------------------------------------------------------
PARTICLE_DTYPE = np.dtype([("x", "f4"), ("y", "f4"), ("z", "f4"), ("u", "f4"), ("v", "f4"), ("w", "f4"), ("E", "f4"),
                           ("particle", "i4")])  # layout of mc_particle (include/mc.h)


def phase_space(n, seed=1, field=(6.0, 6.0), ssd=100.0, z=0.0, fractions=(0.90, 0.08, 0.02), e_max=6.0):
    """Synthetic phase-space list in the plane z: a divergent 6 MV-like beam (PAPER.md:84 names phase-space files as a
    source; none ships with the paper).  Photons with the triangular spectrum of config 3, contaminant electrons
    (uniform 0.3..e_max MeV) and a few positrons; positions uniform over `field`, directions from a point at `ssd`
    with a small Gaussian angular spread.  Input generation only (numpy RNG), no arithmetic of the method."""
    rng = np.random.default_rng(seed)
    p = np.zeros(n, PARTICLE_DTYPE)
    kind = rng.choice(3, size=n, p=np.asarray(fractions) / np.sum(fractions))
    p["particle"] = np.array([PHOTON, ELECTRON, POSITRON], np.int32)[kind]
    x = (rng.random(n) - 0.5) * field[0]
    y = (rng.random(n) - 0.5) * field[1]
    d = np.stack([x + rng.normal(0, 0.5, n), y + rng.normal(0, 0.5, n), np.full(n, ssd)], axis=1)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    p["x"], p["y"], p["z"] = x, y, z
    d32 = d.astype(np.float32).astype(np.float64)
    d32 /= np.linalg.norm(d32, axis=1, keepdims=True)
    p["u"], p["v"], p["w"] = d32[:, 0], d32[:, 1], d32[:, 2]
    # photon energies: triangular pdf 0.25 -> peak at 1.0 -> 0 at 6.0 (inverse CDF), others uniform
    a, c, b = 0.25, 1.0, 6.0
    u = rng.random(n)
    fc = (c - a) / (b - a)
    eg = np.where(u < fc, a + np.sqrt(u * (b - a) * (c - a)), b - np.sqrt((1 - u) * (b - a) * (b - c)))
    ee = 0.3 + rng.random(n) * (e_max - 0.3)
    p["E"] = np.where(kind == 0, eg, ee)
    return p
