"""Shared helpers of the GPU parity tests: oracle-side state from a seeded plasma, comparison
metrics (periodic distance, max-norm relative errors).  No arithmetic of the method."""
import numpy as np

from oracle.psc_oracle import Oracle

PCOLS = ("x", "y", "z", "ux", "uy", "uz", "qw")


def oracle_for(pl, block=(1, 1, 1), scheme=0):
    return Oracle(pl.n, pl.dx, pl.dt, pl.order, pl.q, pl.m, block=block, scheme=scheme)


def oracle_state(pl):
    """fp64 copies of the plasma's fp32 values: dict of particle columns, E, B"""
    st = {k: np.ascontiguousarray(getattr(pl, k).cpu().numpy().astype(np.float64)) for k in PCOLS}
    st["species"] = np.ascontiguousarray(pl.species.cpu().numpy().astype(np.int32))
    st["id"] = np.ascontiguousarray(pl.id.cpu().numpy().astype(np.int32))
    E = np.ascontiguousarray(pl.E.cpu().numpy().astype(np.float64))
    B = np.ascontiguousarray(pl.B.cpu().numpy().astype(np.float64))
    return st, E, B


def gpu_state(sim):
    """dense numpy copy of the cell store through psc_particles_gather (state unchanged): in-cell
    offsets, momenta, qw, species, id and "key", the sort key of the cell each particle is filed
    under"""
    return {k: v.cpu().numpy() for k, v in sim.gather().items() if v is not None}


def gpu_cols(sim, export=True):
    """the particle columns as numpy arrays, dense; export=True: absolute fp32 positions
    ((cell + offset) * dx rounded once, as psc_particles_export gives them); export=False: the
    internal form (in-cell offsets) plus "key".  Neither changes the library's state."""
    if sim.psc.particles_form() == 0:
        return {k: v.cpu().numpy() for k, v in sim.current().items() if v is not None}
    g = sim.gather(absolute=export)
    if export:
        del g["key"]
    return {k: v.cpu().numpy() for k, v in g.items() if v is not None}


def key_to_cell(key, n, block):
    """inverse of the sort key of PAPER.md:593 as the oracle defines it:
    key = block_index * cells_per_block + cell_in_block, both x-fastest"""
    n = np.asarray(n)
    bs = np.asarray(block)
    nb = n // bs
    cpb = int(bs.prod())
    b, l = key // cpb, key % cpb
    bc = (b % nb[0], (b // nb[0]) % nb[1], b // (nb[0] * nb[1]))
    lc = (l % bs[0], (l // bs[0]) % bs[1], l // (bs[0] * bs[1]))
    return [bc[d] * bs[d] + lc[d] for d in range(3)]


def positions_f64(st, pl, block=(0, 0, 0)):
    """fp64 positions (cell + offset) * dx of a gpu_state -- no export rounding; invariant
    coordinates are returned as stored"""
    cells = key_to_cell(st["key"].astype(np.int64), pl.n, library_block(pl.n, block))
    out = []
    for d, c in enumerate(("x", "y", "z")):
        if c not in st:
            out.append(np.zeros(len(st["key"])))
            continue
        o = st[c].astype(np.float64)
        out.append(np.ascontiguousarray(o if pl.n[d] == 1 else (cells[d] + o) * pl.dx[d]))
    return out


def gpu_positions_f64(sim, block=(0, 0, 0)):
    """positions of the current particles in fp64 from the internal form"""
    assert sim.psc.particles_form() == 1
    return positions_f64(gpu_state(sim), sim.plasma, block)


def order_by_id(got_id, ref_id):
    """index array o with got_id[o] == ref_id: the push writes every cell's segment with the
    stayers in front and the leavers behind, so lists are compared particle by particle via id"""
    pos = np.empty(len(got_id), dtype=np.int64)
    pos[got_id] = np.arange(len(got_id))
    o = pos[ref_id]
    assert np.array_equal(got_id[o], ref_id)
    return o


def periodic_dist(a, b, L):
    d = np.abs(a.astype(np.float64) - b.astype(np.float64))
    return np.minimum(d, L - d)


def rel_maxnorm(got, ref):
    """max |got - ref| / max |ref| per leading component -> the largest of them"""
    worst = 0.0
    for c in range(ref.shape[0]):
        den = np.abs(ref[c]).max()
        err = np.abs(got[c].astype(np.float64) - ref[c]).max()
        if den == 0.0:
            assert err == 0.0, "component %d: reference is identically zero, got %g" % (c, err)
            continue
        worst = max(worst, err / den)
    return worst


def rel_fieldnorm(got, ref):
    """max |got - ref| over all components / max |ref| over all components: the north_star's
    'relative to the field's max-norm' read literally (a vector field has one max-norm)"""
    den = np.abs(ref).max()
    err = np.abs(got.astype(np.float64) - ref).max()
    if den == 0.0:
        assert err == 0.0
        return 0.0
    return err / den


def smooth_fields(pl, amp, seed):
    """seeded smooth (few-mode) periodic E and B of amplitude ~amp on the plasma's grid, fp32,
    written into pl.E / pl.B (inputs only -- shared by both paths)"""
    import torch

    rng = np.random.default_rng(seed)
    nx, ny, nz = pl.n
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    out = []
    for _ in range(2):
        F = np.zeros((3, nz, ny, nx))
        for c in range(3):
            for _m in range(3):
                mx = rng.integers(0, 3) if nx > 1 else 0
                my = rng.integers(0, 3) if ny > 1 else 0
                mz = rng.integers(0, 3) if nz > 1 else 0
                ph = rng.uniform(0, 2 * np.pi)
                F[c] += rng.normal() * np.cos(2 * np.pi * (mx * i / nx + my * j / ny + mz * k / nz) + ph)
        out.append(torch.from_numpy((amp * F / 3.0).astype(np.float32)))
    pl.E, pl.B = out[0], out[1]
    return pl


def library_block(n, block=(0, 0, 0)):
    """the block the library uses for a requested `block` (include/psc.h: 0 = default: 8 cells in
    2-d, 4 in 3-d, halved until it divides n; 1 along invariant directions)"""
    is3d = all(v > 1 for v in n)
    out = []
    for d in range(3):
        b = block[d]
        if n[d] == 1:
            b = 1
        elif b == 0:
            b = 4 if is3d else 8
            while n[d] % b:
                b //= 2
        out.append(b)
    return tuple(out)


def oracle_sorted_state(pl, block):
    """the seeded plasma permuted by the ORACLE's stable cell sort: fp32 columns (dict)"""
    orc = oracle_for(pl, block=library_block(pl.n, block))
    cols = {k: getattr(pl, k).cpu().numpy() for k in PCOLS + ("species", "id")}
    _, _, perm, _ = orc.sort(cols["x"], cols["y"], cols["z"])
    return {k: np.ascontiguousarray(v[perm]) for k, v in cols.items()}
