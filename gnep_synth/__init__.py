"""Seeded synthetic Sb-Te-shaped inputs for the GNEP hot path (BASELINE.json `configs` 0-4).

This module serves BOTH the fp64 oracle (tests) and the CUDA path (tests, bench) and therefore holds
none of the method's arithmetic: no basis functions, no descriptors, no network, no loss.  It only
draws structures (cells, positions, species), parameter vectors and label noise from counter-based
streams (numpy Philox keyed by (seed_c, stream)), so that any structure can be regenerated on its own.

The recipe is the one of SURVEY.md section 8(d).2 (restated in DESIGN.md).  The inputs stand in for the
paper's Sb-Te DFT training set, which is not available.  All positions / cells / parameters are
rounded to fp32-representable values so that the oracle (fp64) and the GPU path (fp32 parameters) start
from identical numbers.
"""
import numpy as np

MASTER_SEED = 250700528
DENSITY = 0.030          # atoms / A^3 (configs 2-4 liquids)
A_ROCKSALT = 6.1         # A
RSA_DMIN = 2.4           # A

_STREAM_PARAMS_STUDENT = (1 << 40) + 1
_STREAM_PARAMS_TEACHER = (1 << 40) + 2
_STREAM_NOISE = (1 << 40) + 3
_STREAM_SIZES = (1 << 40) + 4
_STREAM_SPECIES = (1 << 40) + 5


def _base(nr, kr, rcr, na, ka, rca, four, nn):
    return dict(n_species=2, n_radial=nr, n_basis_radial=kr, rc_radial=rcr, n_angular=na,
                n_basis_angular=ka, rc_angular=rca, l_max=4, use_4body=four, n_neurons=nn,
                lambda_e=1.0, lambda_f=1.0, lambda_v=0.1, lambda_2=1e-4, loss_mode=0)


# n_max_X = m  ->  m+1 functions; "K basis functions" -> K functions
MODEL_SPECS = {
    0: _base(5, 8, 6.0, 5, 6, 4.0, False, 10),
    1: _base(9, 12, 7.0, 7, 8, 4.5, True, 30),
    2: _base(9, 12, 7.0, 7, 8, 4.5, True, 50),
    3: _base(11, 12, 7.0, 9, 8, 5.0, True, 80),
    4: _base(11, 12, 8.0, 9, 8, 5.0, True, 100),
}
N_STRUCTS = {0: 4, 1: 100, 2: 200, 3: 1000, 4: 2000}
WORKLOAD_NAMES = {0: "cfg0-tiny-sc", 1: "cfg1-rocksalt-100x216", 2: "cfg2-liquid-200x250",
                  3: "cfg3-mixed-1000", 4: "cfg4-liquid-2000"}


def n_descriptors(spec):
    return (spec["n_radial"] + spec["n_angular"] * spec["l_max"] + (spec["n_angular"] if spec["use_4body"] else 0)
            + (spec["n_angular"] if spec.get("use_5body") else 0))


def n_params(spec):
    T = spec["n_species"]
    nd = n_descriptors(spec)
    return (T * T * spec["n_radial"] * spec["n_basis_radial"] + T * T * spec["n_angular"] * spec["n_basis_angular"]
            + T * (nd * spec["n_neurons"] + 2 * spec["n_neurons"] + 1))


def _rng(config, stream):
    return np.random.Generator(np.random.Philox(key=[MASTER_SEED + config, int(stream)]))


def _f32(a):
    return np.asarray(a, dtype=np.float32).astype(np.float64)


def _finalize(pos, cell):
    """Wrap into the cell, keep fractional coordinates in [1e-6, 1-1e-6], round to fp32 values."""
    cell = _f32(cell)
    frac = pos @ np.linalg.inv(cell)
    frac = frac - np.floor(frac)
    frac = np.clip(frac, 1e-6, 1.0 - 1e-6)
    return _f32(frac @ cell), cell


def _strain(rng):
    e = rng.uniform(-0.03, 0.03, size=6)
    return np.array([[e[0], e[3], e[5]], [e[3], e[1], e[4]], [e[5], e[4], e[2]]])


def _rsa_cubic(rng, n, L):
    """Random sequential insertion with periodic minimum distance RSA_DMIN (candidate order = draw order)."""
    from scipy.spatial import cKDTree
    acc = np.zeros((0, 3))
    while len(acc) < n:
        need = n - len(acc)
        cand = rng.uniform(0.0, L, size=(max(16, 2 * need), 3))
        cand = np.minimum(cand, np.nextafter(L, 0.0))
        if len(acc):
            near = cKDTree(acc, boxsize=L).query_ball_point(cand, RSA_DMIN - 1e-12, return_length=True)
            cand = cand[near == 0]
        if len(cand) == 0:
            continue
        pairs = cKDTree(cand, boxsize=L).query_pairs(RSA_DMIN - 1e-12, output_type="ndarray")
        ok = np.ones(len(cand), dtype=bool)
        if len(pairs):
            lo = np.minimum(pairs[:, 0], pairs[:, 1]); hi = np.maximum(pairs[:, 0], pairs[:, 1])
            order = np.lexsort((lo, hi))
            for a, b in zip(lo[order], hi[order]):     # sequential insertion: later loses to earlier accepted
                if ok[a] and ok[b]:
                    ok[b] = False
        cand = cand[ok][:need]
        acc = np.concatenate([acc, cand], axis=0)
    return acc


def _sc_sites(nx, ny, nz, spacing):
    g = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij"), axis=-1)
    return g.reshape(-1, 3).astype(np.float64) * spacing


def _species_exact(rng, n, frac_sb):
    t = np.ones(n, dtype=np.int32)                     # 1 = Te
    k = int(round(frac_sb * n))
    t[rng.permutation(n)[:k]] = 0                      # 0 = Sb
    return t


def _crystal(rng, nx, ny, nz, vacancy=0.0):
    sp = A_ROCKSALT / 2.0
    pos = _sc_sites(2 * nx, 2 * ny, 2 * nz, sp)
    cell = np.diag([nx * A_ROCKSALT, ny * A_ROCKSALT, nz * A_ROCKSALT]).astype(np.float64)
    types = _species_exact(rng, len(pos), 0.4)
    if vacancy > 0.0:
        keep = np.sort(rng.permutation(len(pos))[int(round(vacancy * len(pos))):])
        pos, types = pos[keep], types[keep]
    dfm = np.eye(3) + _strain(rng)
    pos = (pos + rng.normal(0.0, 0.1, size=pos.shape)) @ dfm
    cell = cell @ dfm
    return pos, cell, types


def _liquid(rng, n):
    L = float(np.float32((n / DENSITY) ** (1.0 / 3.0)))
    pos = _rsa_cubic(rng, n, L)
    x = rng.uniform(0.2, 0.6)
    types = _species_exact(rng, n, x)
    return pos, np.diag([L, L, L]), types


_SUPERCELLS = [(a, b, c) for a in range(1, 9) for b in range(1, 9) for c in range(1, 9)
               if 64 <= 8 * a * b * c <= 512 and max(a, b, c) <= 2 * min(a, b, c)]


def make_structure(config, s):
    """Structure s of config `config`: (positions (n,3) f64, cell (3,3) f64 rows a,b,c, types (n,) i32)."""
    rng = _rng(config, s)
    if config == 0:
        L = 12.4
        pos = _sc_sites(4, 4, 4, 3.1) + rng.uniform(-0.3, 0.3, size=(64, 3))
        types = (rng.uniform(size=64) < 0.5).astype(np.int32)
        cell = np.diag([L, L, L])
    elif config == 1:
        pos, cell, types = _crystal(rng, 3, 3, 3)
    elif config == 2:
        pos, cell, types = _liquid(rng, 250)
    elif config == 3:
        kind = s % 3
        if kind == 1:
            pos, cell, types = _liquid(rng, int(rng.integers(64, 513)))
        else:
            nx, ny, nz = _SUPERCELLS[int(rng.integers(0, len(_SUPERCELLS)))]
            pos, cell, types = _crystal(rng, nx, ny, nz, vacancy=0.05 if kind == 2 else 0.0)
    elif config == 4:
        pos, cell, types = _liquid(rng, int(rng.integers(96, 1001)))
    else:
        raise ValueError("config must be 0..4")
    pos, cell = _finalize(pos, cell)
    return pos, cell, np.ascontiguousarray(types, dtype=np.int32)


def _make_structure_job(args):
    return make_structure(*args)


def make_batch(config, n_structs=None, first=0, workers=0):
    """Structures first .. first+n_structs-1 of a config, concatenated.  Every structure depends only on
    (config, s), so `workers` > 1 (processes) changes nothing but the wall time.

    Returns dict(atom_offsets i32 [S+1], positions f64 [N,3], cells f64 [S,9], types i32 [N])."""
    S = N_STRUCTS[config] if n_structs is None else int(n_structs)
    jobs = [(config, s) for s in range(first, first + S)]
    if workers and workers > 1 and S >= 4 * workers:
        import multiprocessing as mp
        with mp.get_context("fork").Pool(workers) as pool:
            res = pool.map(_make_structure_job, jobs, chunksize=max(1, S // (8 * workers)))
    else:
        res = [make_structure(*j) for j in jobs]
    P, Cc, Tt, off = [], [], [], [0]
    for p, c, t in res:
        P.append(p); Cc.append(c.reshape(9)); Tt.append(t); off.append(off[-1] + len(p))
    return dict(atom_offsets=np.asarray(off, dtype=np.int32),
                positions=np.concatenate(P, axis=0) if P else np.zeros((0, 3)),
                cells=np.stack(Cc, axis=0) if Cc else np.zeros((0, 9)),
                types=np.concatenate(Tt, axis=0) if Tt else np.zeros((0,), dtype=np.int32))


def relabel_species(types, n_species, config):
    """Species ids for a model with `n_species` != 2 kinds of atoms on the same sites (test inputs for T = 1, 3, 4):
    all zeros for one species, otherwise i.i.d. uniform draws from [0, n_species) on a stream of their own."""
    n = len(types)
    if n_species == 1:
        return np.zeros(n, dtype=np.int32)
    return _rng(config, _STREAM_SPECIES).integers(0, n_species, size=n).astype(np.int32)


def draw_params(spec, config, which="student"):
    """Flat parameter vector (layout of include/gnep.h): c ~ U(-1,1); W0,b0 ~ N(0,1/N_des); w1,b1 ~ N(0,1/Nn)."""
    rng = _rng(config, _STREAM_PARAMS_STUDENT if which == "student" else _STREAM_PARAMS_TEACHER)
    T, nd, nn = spec["n_species"], n_descriptors(spec), spec["n_neurons"]
    parts = [rng.uniform(-1.0, 1.0, size=T * T * spec["n_radial"] * spec["n_basis_radial"]),
             rng.uniform(-1.0, 1.0, size=T * T * spec["n_angular"] * spec["n_basis_angular"])]
    for _ in range(T):
        parts.append(rng.normal(0.0, 1.0 / np.sqrt(nd), size=nn * nd))     # W0
        parts.append(rng.normal(0.0, 1.0 / np.sqrt(nd), size=nn))          # b0
        parts.append(rng.normal(0.0, 1.0 / np.sqrt(nn), size=nn))          # w1
        parts.append(rng.normal(0.0, 1.0 / np.sqrt(nn), size=1))           # b1
    return _f32(np.concatenate(parts))


def add_label_noise(config, atom_offsets, E, F, W):
    """Teacher labels + noise: sigma_E = 1 meV/atom, sigma_F = 20 meV/A, no virial noise."""
    rng = _rng(config, _STREAM_NOISE)
    ns = np.diff(np.asarray(atom_offsets)).astype(np.float64)
    E = np.asarray(E, dtype=np.float64) + ns * rng.normal(0.0, 1e-3, size=len(ns))
    F = np.asarray(F, dtype=np.float64) + rng.normal(0.0, 0.02, size=np.shape(F))
    return E, F, np.asarray(W, dtype=np.float64).copy()


def q_scale_from(q):
    """Fixed, non-trainable input scaling 1/(max-min) per descriptor column, fp32 values."""
    q = np.asarray(q, dtype=np.float64)
    rng_ = q.max(axis=0) - q.min(axis=0)
    s = np.where(rng_ > 0, 1.0 / np.where(rng_ > 0, rng_, 1.0), 1.0)
    return _f32(s)
