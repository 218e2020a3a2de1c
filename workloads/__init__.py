"""Seeded synthetic inputs shared by the CPU oracle and the CUDA path.

This module holds NONE of the method's arithmetic (no DG operator, no flux, no
Riemann solver, no rate law).  It only builds *inputs*: meshes (node coordinates
+ connectivity lists in the layout of include/marut.h), initial fields shaped
like the paper's workloads, and the synthetic thermochemical tables of config 5.
All random draws come from a counter-based generator (splitmix64 of
(seed, stream, index) -> uniform [0,1)), so the same numbers reach both sides.

The recipe for every config is stated in DESIGN.md section 5.

Layouts (row-major, last index fastest; n = N+1, node = i + n*(j + n*k)):
  node_xyz [n_elem][dim][n^dim]  float64
  u        [n_elem][n_var][n^dim] float64, v = rho_1..rho_ns, rho*u_1..rho*u_d, E
  iface    [n_iface][5]  int32 = eL,fL,eR,fR,orient   (face f = 2*l + side)
  mortar   [n_mortar][6] int32 = eC,fC,eF_lo,eF_up,fF,orient   (2-D only)
  bface    [n_bface][3]  int32 = e,f,bc_id ; bc_state [n_bc][n_var] float64
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED = 20260526
EULER, NAVIER_STOKES, REACTING_EULER = 0, 1, 2
R_UNIVERSAL = 8.31446261815324


# ----------------------------------------------------------------------------
# counter-based random numbers
# ----------------------------------------------------------------------------
def _splitmix64(x: np.ndarray) -> np.ndarray:
    x = (x + np.uint64(0x9E3779B97F4A7C15)).astype(np.uint64)
    z = x
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def uniform(seed: int, stream: int, index) -> np.ndarray:
    """uniform [0,1) doubles, a pure function of (seed, stream, index)."""
    with np.errstate(over="ignore"):
        idx = np.asarray(index, dtype=np.uint64)
        k = _splitmix64(np.uint64(seed) + _splitmix64(np.uint64(stream) + np.zeros_like(idx)))
        z = _splitmix64(k ^ _splitmix64(idx))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# ----------------------------------------------------------------------------
# Legendre-Gauss-Lobatto abscissae (library routine: numpy's Legendre class);
# only used to place the isoparametric mesh nodes the descriptor asks for.
# ----------------------------------------------------------------------------
def lgl_points(N: int) -> np.ndarray:
    from numpy.polynomial import legendre as L

    c = np.zeros(N + 1)
    c[N] = 1.0
    inner = np.sort(L.legroots(L.legder(c))) if N > 1 else np.zeros(0)
    x = np.concatenate([[-1.0], inner, [1.0]])
    x = 0.5 * (x - x[::-1])  # exact antisymmetry
    return x


# ----------------------------------------------------------------------------
# mesh container
# ----------------------------------------------------------------------------
@dataclass
class Mech:
    names: list
    W: np.ndarray  # [ns] kg/mol
    nasa: np.ndarray  # [ns][2][7]
    T_mid: float
    nu_r: np.ndarray  # [nr][ns] int32
    nu_p: np.ndarray  # [nr][ns] int32
    A: np.ndarray
    b: np.ndarray
    Ea: np.ndarray

    @property
    def ns(self):
        return len(self.W)

    @property
    def nr(self):
        return len(self.A)


@dataclass
class Mesh:
    dim: int
    N: int
    node_xyz: np.ndarray
    iface: np.ndarray
    mortar: np.ndarray = field(default_factory=lambda: np.zeros((0, 6), np.int32))
    bface: np.ndarray = field(default_factory=lambda: np.zeros((0, 3), np.int32))
    bc_state: np.ndarray = field(default_factory=lambda: np.zeros((0, 0)))
    physics: int = EULER
    gamma: float = 1.4
    mu: float = 0.0
    Pr: float = 0.72
    mech: Mech | None = None
    volume_form: int = 0   # 0: standard strong-form volume integral (eq. 9); 1: entropy-stable split form (eq. 10)
    info: dict = field(default_factory=dict)

    @property
    def n_elem(self):
        return self.node_xyz.shape[0]

    @property
    def n(self):
        return self.N + 1

    @property
    def nn(self):
        return self.n ** self.dim

    @property
    def n_var(self):
        ns = self.mech.ns if self.physics == REACTING_EULER else 1
        return ns + self.dim + 1

    @property
    def n_dof(self):
        return self.n_elem * self.nn * self.n_var


# ----------------------------------------------------------------------------
# Cartesian periodic meshes (configs 1, 2, 3, 5)
# ----------------------------------------------------------------------------
def _morton_order(counts):
    """element order along a Morton (Z) curve; falls back to lexicographic when
    the counts are not equal powers of two."""
    dim = len(counts)
    idx = np.indices(counts[::-1]).reshape(dim, -1)[::-1]  # idx[c] = coordinate c, x fastest
    c0 = counts[0]
    pow2 = all(c == c0 for c in counts) and (c0 & (c0 - 1)) == 0
    if not pow2:
        return idx
    bits = max(1, int(c0).bit_length() - 1)
    key = np.zeros(idx.shape[1], dtype=np.int64)
    for b in range(bits):
        for c in range(dim):
            key |= ((idx[c] >> b) & 1).astype(np.int64) << (b * dim + c)
    perm = np.argsort(key, kind="stable")
    return idx[:, perm]


def cartesian_mesh(dim, N, counts, lo, hi, order="morton", warp=None, periodic=True) -> Mesh:
    """uniform box mesh, all directions periodic; `warp(X) -> x` is applied to the
    global coordinates of every LGL node (so shared faces coincide)."""
    counts = tuple(int(c) for c in counts)
    assert len(counts) == dim and periodic
    xi = lgl_points(N)
    n = N + 1
    if order == "morton":
        eidx = _morton_order(counts)
    else:
        eidx = np.indices(counts[::-1]).reshape(dim, -1)[::-1]
    ne = eidx.shape[1]
    h = [(hi[c] - lo[c]) / counts[c] for c in range(dim)]
    # element id lookup
    lut = np.empty(counts[::-1], dtype=np.int64)
    lut[tuple(eidx[c] for c in range(dim - 1, -1, -1))] = np.arange(ne)
    # node coordinates
    ref = np.indices((n,) * dim).reshape(dim, -1)[::-1]  # ref[c][node] = index along c, i fastest
    frac = (xi[ref] + 1.0) / 2.0  # [dim][nn], exactly 0 and 1 at the ends
    X = np.empty((ne, dim, n ** dim))
    for c in range(dim):
        X[:, c, :] = lo[c] + (eidx[c][:, None] + frac[c][None, :]) * h[c]
    if warp is not None:
        X = warp(X)
    # interfaces: each element owns its +side face in every direction
    ifaces = []
    for l in range(dim):
        nb = [eidx[c].copy() for c in range(dim)]
        nb[l] = (nb[l] + 1) % counts[l]
        eR = lut[tuple(nb[c] for c in range(dim - 1, -1, -1))]
        blk = np.empty((ne, 5), dtype=np.int32)
        blk[:, 0] = np.arange(ne)
        blk[:, 1] = 2 * l + 1
        blk[:, 2] = eR
        blk[:, 3] = 2 * l
        blk[:, 4] = 0
        ifaces.append(blk)
    iface = np.ascontiguousarray(np.concatenate(ifaces, axis=0))
    m = Mesh(dim=dim, N=N, node_xyz=np.ascontiguousarray(X), iface=iface)
    m.info = dict(counts=counts, lo=tuple(lo), hi=tuple(hi), h=tuple(h), order=order)
    return m


def open_direction(mesh: Mesh, axis=0, bc_lo=0, bc_hi=1) -> Mesh:
    """turn the periodic wrap-around interfaces of a Cartesian mesh in direction `axis` into boundary faces
    (boundary id bc_lo on the low side, bc_hi on the high side); rows are appended to mesh.bface"""
    xc = mesh.node_xyz[:, axis, :].mean(axis=1)
    first, last = np.isclose(xc, xc.min()), np.isclose(xc, xc.max())
    wrap = (mesh.iface[:, 1] == 2 * axis + 1) & last[mesh.iface[:, 0]] & first[mesh.iface[:, 2]]
    assert wrap.sum() == last.sum() > 0
    w = mesh.iface[wrap]
    new = np.concatenate([np.stack([w[:, 0], w[:, 1], np.full(len(w), bc_hi, np.int32)], axis=1),
                          np.stack([w[:, 2], w[:, 3], np.full(len(w), bc_lo, np.int32)], axis=1)]).astype(np.int32)
    mesh.bface = np.ascontiguousarray(np.concatenate([mesh.bface.reshape(-1, 3), new]).astype(np.int32))
    mesh.iface = np.ascontiguousarray(mesh.iface[~wrap])
    return mesh


def octree_box_mesh(N, K=4, lo=(0.0, 0.0, 0.0), hi=(1.0, 1.0, 1.0), refine=None) -> Mesh:
    """3-D periodic box of K^3 cells, the cells selected by `refine(ix, iy, iz) -> bool` (default: ix < K/2) split once
    into 2x2x2 children: conforming faces between cells of equal size, 4:1 mortar faces (rows of 8 ints:
    eC, fC, eF_00, eF_10, eF_01, eF_11, fF, 0; eF_{s0 s1} = the fine element on half s0 / s1 of the coarse face's first /
    second face-local direction) between a cell and a split neighbour.  Affine elements."""
    if refine is None:
        refine = lambda ix, iy, iz: ix < K // 2
    n = N + 1
    xi = lgl_points(N)
    h = [(hi[c] - lo[c]) / K for c in range(3)]
    ref = np.indices((n, n, n)).reshape(3, -1)[::-1]
    frac = (xi[ref] + 1.0) / 2.0
    split = {(ix, iy, iz): bool(refine(ix, iy, iz)) for ix in range(K) for iy in range(K) for iz in range(K)}
    ids, X = {}, []

    def add(key, origin, size):
        ids[key] = len(X)
        X.append(np.stack([origin[c] + frac[c] * size[c] for c in range(3)]))

    for iz in range(K):
        for iy in range(K):
            for ix in range(K):
                cell = (ix, iy, iz)
                o = [lo[c] + cell[c] * h[c] for c in range(3)]
                if not split[cell]:
                    add((cell, None), o, h)
                else:
                    for cz in range(2):
                        for cy in range(2):
                            for cx in range(2):
                                ch = (cx, cy, cz)
                                add((cell, ch), [o[c] + 0.5 * h[c] * ch[c] for c in range(3)], [0.5 * hc for hc in h])
    iface, mortar = [], []

    def child(l, side, s0, s1):
        rest = [c for c in range(3) if c != l]
        ch = [0, 0, 0]
        ch[l], ch[rest[0]], ch[rest[1]] = side, s0, s1
        return tuple(ch)

    for cell in split:
        for l in range(3):
            nb = list(cell)
            nb[l] = (nb[l] + 1) % K
            nb = tuple(nb)
            if split[cell]:                                   # faces between the children of this cell
                for s1 in range(2):
                    for s0 in range(2):
                        iface.append((ids[(cell, child(l, 0, s0, s1))], 2 * l + 1, ids[(cell, child(l, 1, s0, s1))], 2 * l, 0))
            if not split[cell] and not split[nb]:
                iface.append((ids[(cell, None)], 2 * l + 1, ids[(nb, None)], 2 * l, 0))
            elif split[cell] and split[nb]:
                for s1 in range(2):
                    for s0 in range(2):
                        iface.append((ids[(cell, child(l, 1, s0, s1))], 2 * l + 1, ids[(nb, child(l, 0, s0, s1))], 2 * l, 0))
            elif not split[cell]:                             # coarse cell, split neighbour on its + side
                fine = [ids[(nb, child(l, 0, s0, s1))] for s1 in range(2) for s0 in range(2)]
                mortar.append((ids[(cell, None)], 2 * l + 1, *fine, 2 * l, 0))
            else:                                             # split cell, coarse neighbour on its + side
                fine = [ids[(cell, child(l, 1, s0, s1))] for s1 in range(2) for s0 in range(2)]
                mortar.append((ids[(nb, None)], 2 * l, *fine, 2 * l + 1, 0))
    m = Mesh(dim=3, N=N, node_xyz=np.ascontiguousarray(np.stack(X)), iface=np.ascontiguousarray(np.array(iface, dtype=np.int32)),
             mortar=np.ascontiguousarray(np.array(mortar, dtype=np.int32).reshape(-1, 8)))
    m.info = dict(K=K, lo=tuple(lo), hi=tuple(hi), n_split=int(sum(split.values())))
    return m


def _cube_rotations():
    """the 24 proper rotations of the reference cube as (perm, sign): new axis d runs along old axis perm[d], reversed
    where sign[d] < 0"""
    import itertools
    out = []
    for perm in itertools.permutations(range(3)):
        for sign in itertools.product((1, -1), repeat=3):
            M = np.zeros((3, 3))
            for d in range(3):
                M[d, perm[d]] = sign[d]
            if round(np.linalg.det(M)) == 1:
                out.append((perm, sign))
    return out


def face_orientation(n, pairs):
    """3-D orientation code of a conforming face from node pairs ((a0, a1) on the left, (b0, b1) on the right):
    (c0, c1) = (a1, a0) if code & 4 else (a0, a1);  b0 = n-1-c0 if code & 1 else c0;  b1 = n-1-c1 if code & 2 else c1"""
    for code in range(8):
        ok = True
        for (a0, a1), (b0, b1) in pairs:
            c0, c1 = (a1, a0) if code & 4 else (a0, a1)
            if code & 1:
                c0 = n - 1 - c0
            if code & 2:
                c1 = n - 1 - c1
            if (c0, c1) != (b0, b1):
                ok = False
                break
        if ok:
            return code
    raise ValueError("face nodes do not match under any orientation")


def rotate_elements(mesh: Mesh, seed=SEED, frac=0.6):
    """3-D conforming mesh -> the same mesh with the local axes of a seeded subset of elements rotated (one of the 24
    proper rotations each), as an unstructured hexahedral mesh presents them: face numbers and the relative orientation
    of the two sides of an interface change, the geometry does not.  Returns (new mesh, node_map) with
    node_map[e][new_node] = old_node, so that field_new[e, :, :] = field_old[e, :, node_map[e]]."""
    assert mesh.dim == 3 and len(mesh.mortar) == 0
    n, ne = mesh.n, mesh.n_elem
    rots = _cube_rotations()
    pick = uniform(seed, 77, np.arange(ne))
    which = (uniform(seed, 78, np.arange(ne)) * 24).astype(int) % 24
    rot = [rots[which[e]] if pick[e] < frac else ((0, 1, 2), (1, 1, 1)) for e in range(ne)]
    idx = np.indices((n, n, n)).reshape(3, -1)[::-1]              # idx[c][node] = index along axis c, i fastest
    node_map = np.empty((ne, n ** 3), dtype=np.int64)
    new_of_old = np.empty((ne, n ** 3), dtype=np.int64)
    for e in range(ne):
        perm, sign = rot[e]
        # new multi-index (i'_0, i'_1, i'_2) -> old multi-index: old[perm[d]] = i'_d or n-1-i'_d
        old = [None] * 3
        for d in range(3):
            old[perm[d]] = idx[d] if sign[d] > 0 else n - 1 - idx[d]
        node_map[e] = old[0] + n * (old[1] + n * old[2])
        new_of_old[e, node_map[e]] = np.arange(n ** 3)
    X = np.stack([mesh.node_xyz[e][:, node_map[e]] for e in range(ne)])

    def face_of(node_new):
        """(face id, a0, a1) candidates of a node given by its new multi-index"""
        return [node_new % n, (node_new // n) % n, node_new // (n * n)]

    def new_face(e, f_old):
        l, side = f_old // 2, f_old % 2
        perm, sign = rot[e]
        d = perm.index(l)
        return 2 * d + (side if sign[d] > 0 else 1 - side)

    def face_local(e, f_new, node_new):
        ijk = face_of(node_new)
        rest = [c for c in range(3) if c != f_new // 2]
        return int(ijk[rest[0]]), int(ijk[rest[1]])

    def old_face_node(f, a0, a1):
        l, side = f // 2, f % 2
        ijk = [0, 0, 0]
        rest = [c for c in range(3) if c != l]
        ijk[l] = (n - 1) if side else 0
        ijk[rest[0]], ijk[rest[1]] = a0, a1
        return ijk[0] + n * (ijk[1] + n * ijk[2])

    iface = np.empty_like(mesh.iface)
    probes = [(0, 0), (n - 1, 0), (0, n - 1), (1 % n, 0)] if n > 2 else [(0, 0), (1, 0), (0, 1), (1, 1)]
    for q, (eL, fL, eR, fR, orient) in enumerate(mesh.iface):
        assert orient == 0
        fLn, fRn = new_face(eL, fL), new_face(eR, fR)
        pairs = []
        for a0, a1 in probes:
            pL = new_of_old[eL, old_face_node(fL, a0, a1)]
            pR = new_of_old[eR, old_face_node(fR, a0, a1)]
            pairs.append((face_local(eL, fLn, pL), face_local(eR, fRn, pR)))
        iface[q] = (eL, fLn, eR, fRn, face_orientation(n, pairs))
    m = Mesh(dim=3, N=mesh.N, node_xyz=np.ascontiguousarray(X), iface=np.ascontiguousarray(iface), physics=mesh.physics,
             gamma=mesh.gamma, mu=mesh.mu, Pr=mesh.Pr, mech=mesh.mech, volume_form=mesh.volume_form)
    m.info = dict(mesh.info, rotated=int(sum(r != ((0, 1, 2), (1, 1, 1)) for r in rot)))
    return m, node_map


def sine_warp(counts, lo, hi, amp_frac=0.05, k=8, seed=SEED):
    """config 3: x_c = X_c + amp*h * prod_d sin(k X_d + phi_{c,d}), seeded phases."""
    dim = len(counts)
    h = (hi[0] - lo[0]) / counts[0]
    phases = 2.0 * math.pi * uniform(seed, 31, np.arange(dim * dim)).reshape(dim, dim)
    scale = 2.0 * math.pi / (hi[0] - lo[0])  # k waves per domain length

    def warp(X):
        out = X.copy()
        for c in range(dim):
            prod = np.ones_like(X[:, 0, :])
            for d in range(dim):
                prod = prod * np.sin(k * scale * (X[:, d, :] - lo[d]) + phases[c, d])
            out[:, c, :] = X[:, c, :] + amp_frac * h * prod
        return out

    return warp


# ----------------------------------------------------------------------------
# 2:1-balanced quadtree mesh (config 4)
# ----------------------------------------------------------------------------
def quadtree_mesh(N, base=(128, 32), lo=(0.0, 0.0), hi=(4.0, 1.0), max_level=3, band=0.15,
                  jitter=0.0, seed=SEED) -> Mesh:
    """static AMR mesh refined `max_level` levels where |x - x_s(y)| < band,
    x_s(y) = 1 + 0.2 sin(2 pi y); then face-2:1 balanced; leaves
    ordered by base cell then Morton.  y periodic, x bounded:
    left boundary bc_id 0, right boundary bc_id 1."""
    Bx, By = base
    h0x, h0y = (hi[0] - lo[0]) / Bx, (hi[1] - lo[1]) / By
    row_w = band * (1.0 + jitter * (2.0 * uniform(seed, 41, np.arange(By)) - 1.0))

    def wants(l, ix, iy):
        hx, hy = h0x / (1 << l), h0y / (1 << l)
        w = row_w[(iy >> l) % By]
        for sy in (0.0, 0.5, 1.0):
            y = lo[1] + (iy + sy) * hy
            xs = 1.0 + 0.2 * math.sin(2.0 * math.pi * y)
            x0, x1 = lo[0] + ix * hx, lo[0] + (ix + 1) * hx
            d = 0.0 if x0 <= xs <= x1 else min(abs(x0 - xs), abs(x1 - xs))
            if d < w:
                return True
        return False

    leaves = set()
    stack = [(0, ix, iy) for iy in range(By) for ix in range(Bx)]
    while stack:
        l, ix, iy = stack.pop()
        if l < max_level and wants(l, ix, iy):
            for dy in (0, 1):
                for dx in (0, 1):
                    stack.append((l + 1, 2 * ix + dx, 2 * iy + dy))
        else:
            leaves.add((l, ix, iy))

    def find_leaf(l, ix, iy):
        """leaf that is the cell (l,ix,iy) or one of its ancestors; None if the cell is subdivided"""
        for k in range(l + 1):
            c = (l - k, ix >> k, iy >> k)
            if c in leaves:
                return c
        return None

    def neighbor(l, ix, iy, d):
        nx, ny = Bx << l, By << l
        jx, jy = ix + (1 if d == 1 else -1 if d == 0 else 0), iy + (1 if d == 3 else -1 if d == 2 else 0)
        if jx < 0 or jx >= nx:
            return None
        return (l, jx, jy % ny)

    # face 2:1 balance
    changed = True
    while changed:
        changed = False
        for (l, ix, iy) in list(leaves):
            if (l, ix, iy) not in leaves:
                continue
            for d in range(4):
                nb = neighbor(l, ix, iy, d)
                if nb is None:
                    continue
                lf = find_leaf(*nb)
                if lf is not None and lf[0] < l - 1:
                    leaves.discard(lf)
                    for dy in (0, 1):
                        for dx in (0, 1):
                            leaves.add((lf[0] + 1, 2 * lf[1] + dx, 2 * lf[2] + dy))
                    changed = True

    def sort_key(c):
        l, ix, iy = c
        bx, by = ix >> l, iy >> l
        sx, sy = (ix - (bx << l)) << (max_level - l), (iy - (by << l)) << (max_level - l)
        mort = 0
        for b in range(max_level):
            mort |= ((sx >> b) & 1) << (2 * b) | ((sy >> b) & 1) << (2 * b + 1)
        return (by * Bx + bx, mort)

    order = sorted(leaves, key=sort_key)
    eid = {c: i for i, c in enumerate(order)}
    ne = len(order)

    xi = lgl_points(N)
    n = N + 1
    ref = np.indices((n, n)).reshape(2, -1)[::-1]
    frac = (xi[ref] + 1.0) / 2.0
    lev = np.array([c[0] for c in order])
    ixs = np.array([c[1] for c in order])
    iys = np.array([c[2] for c in order])
    hx, hy = h0x / (1 << lev), h0y / (1 << lev)
    X = np.empty((ne, 2, n * n))
    X[:, 0, :] = lo[0] + (ixs[:, None] + frac[0][None, :]) * hx[:, None]
    X[:, 1, :] = lo[1] + (iys[:, None] + frac[1][None, :]) * hy[:, None]

    iface, mortar, bface = [], [], []
    opp = {0: 1, 1: 0, 2: 3, 3: 2}
    for c in order:
        l, ix, iy = c
        e = eid[c]
        for d in range(4):
            nb = neighbor(l, ix, iy, d)
            if nb is None:
                bface.append((e, d, 0 if d == 0 else 1))
                continue
            if nb in leaves:
                if d in (1, 3):  # each conforming interface once, from its - side element
                    iface.append((e, d, eid[nb], opp[d], 0))
                continue
            if find_leaf(*nb) is not None:
                continue  # neighbour is coarser: the mortar is recorded from the coarse side
            # neighbour is subdivided: two fine leaves touch this face
            _, jx, jy = nb
            if d == 1:
                kids = [(l + 1, 2 * jx, 2 * jy), (l + 1, 2 * jx, 2 * jy + 1)]
            elif d == 0:
                kids = [(l + 1, 2 * jx + 1, 2 * jy), (l + 1, 2 * jx + 1, 2 * jy + 1)]
            elif d == 3:
                kids = [(l + 1, 2 * jx, 2 * jy), (l + 1, 2 * jx + 1, 2 * jy)]
            else:
                kids = [(l + 1, 2 * jx, 2 * jy + 1), (l + 1, 2 * jx + 1, 2 * jy + 1)]
            assert kids[0] in leaves and kids[1] in leaves, "mesh is not 2:1 balanced"
            mortar.append((e, d, eid[kids[0]], eid[kids[1]], opp[d], 0))

    m = Mesh(dim=2, N=N, node_xyz=np.ascontiguousarray(X),
             iface=np.array(iface, dtype=np.int32).reshape(-1, 5),
             mortar=np.array(mortar, dtype=np.int32).reshape(-1, 6),
             bface=np.array(bface, dtype=np.int32).reshape(-1, 3))
    m.info = dict(base=base, lo=lo, hi=hi, max_level=max_level, band=band, levels=np.bincount(lev, minlength=max_level + 1).tolist(),
                  h_fine=h0x / (1 << max_level))
    return m


# ----------------------------------------------------------------------------
# initial fields
# ----------------------------------------------------------------------------
def _cons_from_prim(rho, vel, p, gamma):
    ke = 0.5 * rho * sum(v * v for v in vel)
    E = p / (gamma - 1.0) + ke
    return np.stack([rho] + [rho * v for v in vel] + [E], axis=1)


def isentropic_vortex(mesh: Mesh, t=0.0, beta=5.0, center=(5.0, 5.0), L=10.0):
    """config 1 (free stream rho=u=v=p=1); exact solution = translation by (t,t), periodic in L."""
    g = mesh.gamma
    x = mesh.node_xyz[:, 0, :] - center[0] - t
    y = mesh.node_xyz[:, 1, :] - center[1] - t
    x = x - L * np.round(x / L)
    y = y - L * np.round(y / L)
    r2 = x * x + y * y
    f = beta / (2.0 * math.pi) * np.exp(0.5 * (1.0 - r2))
    u = 1.0 - f * y
    v = 1.0 + f * x
    T = 1.0 - (g - 1.0) * beta * beta / (8.0 * g * math.pi ** 2) * np.exp(1.0 - r2)
    rho = T ** (1.0 / (g - 1.0))
    p = rho ** g
    return np.ascontiguousarray(_cons_from_prim(rho, [u, v], p, g))


def taylor_green(mesh: Mesh, mach=0.1, noise=0.0, seed=SEED):
    """configs 2, 3: eq. 28 with A = 1 on [0, 2 pi]^3."""
    g = mesh.gamma
    x, y, z = (mesh.node_xyz[:, c, :] for c in range(3))
    rho = np.ones_like(x)
    u = np.sin(x) * np.cos(y) * np.cos(z)
    v = -np.cos(x) * np.sin(y) * np.cos(z)
    w = np.zeros_like(x)
    p = 1.0 / (g * mach * mach) + (np.cos(2 * x) * np.cos(2 * z) + 2 * np.cos(2 * y) + 2 * np.cos(2 * x)
                                   + np.cos(2 * y) * np.cos(2 * z)) / 16.0
    if noise > 0.0:
        idx = np.arange(x.size).reshape(x.shape)
        u = u + noise * (2.0 * uniform(seed, 11, idx) - 1.0)
        v = v + noise * (2.0 * uniform(seed, 12, idx) - 1.0)
        w = w + noise * (2.0 * uniform(seed, 13, idx) - 1.0)
    return np.ascontiguousarray(_cons_from_prim(rho, [u, v, w], p, g))


SHOCK_PRE = (1.4, 0.0, 0.0, 1.0)  # Mach-10 normal shock into (rho,u,v,p) = (1.4,0,0,1), a_1 = 1
SHOCK_POST = (8.0, 8.25, 0.0, 116.5)


def shock_states(gamma=1.4):
    def cons(s):
        rho, u, v, p = s
        return np.array([rho, rho * u, rho * v, p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v)])
    return np.stack([cons(SHOCK_POST), cons(SHOCK_PRE)])  # bc_id 0 = left = post, 1 = right = pre


def mach10_shock(mesh: Mesh, half_width):
    """config 4: tanh-regularised normal shock along x_s(y) = 1 + 0.2 sin(2 pi y)."""
    g = mesh.gamma
    x, y = mesh.node_xyz[:, 0, :], mesh.node_xyz[:, 1, :]
    xs = 1.0 + 0.2 * np.sin(2.0 * math.pi * y)
    s = 0.5 * (1.0 + np.tanh((x - xs) / half_width))  # 0 = post-shock (left), 1 = pre-shock (right)
    prim = [SHOCK_POST[k] + (SHOCK_PRE[k] - SHOCK_POST[k]) * s for k in range(4)]
    return np.ascontiguousarray(_cons_from_prim(prim[0], [prim[1], prim[2]], prim[3], g))


# ----------------------------------------------------------------------------
# config 5: synthetic 5-species air mechanism + NASA-7-form tables
# ----------------------------------------------------------------------------
def _nasa7_eval(a, T):
    cp = a[0] + a[1] * T + a[2] * T ** 2 + a[3] * T ** 3 + a[4] * T ** 4
    h = a[0] + a[1] * T / 2 + a[2] * T ** 2 / 3 + a[3] * T ** 3 / 4 + a[4] * T ** 4 / 5 + a[5] / T
    s = a[0] * np.log(T) + a[1] * T + a[2] * T ** 2 / 2 + a[3] * T ** 3 / 3 + a[4] * T ** 4 / 4 + a[6]
    return cp, h, s


def air5_mechanism(seed=SEED) -> Mech:
    """(N2,O2,NO,N,O); 3 dissociations x 5 third bodies + 2 exchanges = 17 reversible
    reactions with SEEDED Arrhenius parameters (BASELINE.json config 5);
    NASA-7-form tables by least squares on rigid-rotor/harmonic-oscillator cp."""
    names = ["N2", "O2", "NO", "N", "O"]
    WN, WO = 14.0067e-3, 15.9994e-3
    W = np.array([2 * WN, 2 * WO, WN + WO, WN, WO])
    theta_v = [3395.0, 2239.0, 2817.0, None, None]
    hf = np.array([0.0, 0.0, 90.29e3, 472.68e3, 249.17e3])  # J/mol at 298.15 K
    s0 = np.array([191.6, 205.1, 210.8, 153.3, 161.1])  # J/(mol K) at 298.15 K
    T_mid = 1000.0
    nasa = np.zeros((5, 2, 7))
    for s in range(5):
        for r, (Ta, Tb) in enumerate([(200.0, T_mid), (T_mid, 10000.0)]):
            T = np.linspace(Ta, Tb, 400)
            if theta_v[s] is None:
                cp = np.full_like(T, 2.5)
            else:
                xx = theta_v[s] / T
                cp = 3.5 + xx * xx * np.exp(xx) / (np.exp(xx) - 1.0) ** 2
            Ts = T / 1000.0  # scaled for conditioning
            V = np.stack([Ts ** k for k in range(5)], axis=1)
            c, *_ = np.linalg.lstsq(V, cp, rcond=None)
            nasa[s, r, :5] = c / np.array([1000.0 ** k for k in range(5)])
        # low range: h(298.15) = hf, s(298.15) = s0
        a = nasa[s, 0]
        _, h, ss = _nasa7_eval(a, 298.15)
        a[5] = (hf[s] / (R_UNIVERSAL * 298.15) - h) * 298.15
        a[6] = s0[s] / R_UNIVERSAL - ss
        # high range: continuity of h and s at T_mid
        _, hl, sl = _nasa7_eval(nasa[s, 0], T_mid)
        b = nasa[s, 1]
        _, hh, sh = _nasa7_eval(b, T_mid)
        b[5] = (hl - hh) * T_mid
        b[6] = sl - sh
    nu_r, nu_p = [], []
    diss = [(0, {3: 2}), (1, {4: 2}), (2, {3: 1, 4: 1})]
    for mol, prod in diss:
        for M in range(5):
            r = np.zeros(5, np.int32)
            p = np.zeros(5, np.int32)
            r[mol] += 1
            r[M] += 1
            p[M] += 1
            for k, c in prod.items():
                p[k] += c
            nu_r.append(r)
            nu_p.append(p)
    for rr, pp in [({0: 1, 4: 1}, {2: 1, 3: 1}), ({3: 1, 1: 1}, {2: 1, 4: 1})]:  # N2+O=NO+N ; N+O2=NO+O
        r = np.zeros(5, np.int32)
        p = np.zeros(5, np.int32)
        for k, c in rr.items():
            r[k] += c
        for k, c in pp.items():
            p[k] += c
        nu_r.append(r)
        nu_p.append(p)
    nr = len(nu_r)
    A = 10.0 ** (12.0 + 10.0 * uniform(seed, 51, np.arange(nr)))
    b = -2.0 * uniform(seed, 52, np.arange(nr))
    Ea = 5.0e4 + 7.0e4 * uniform(seed, 53, np.arange(nr))
    return Mech(names=names, W=W, nasa=np.ascontiguousarray(nasa), T_mid=T_mid,
                nu_r=np.ascontiguousarray(np.array(nu_r, np.int32)), nu_p=np.ascontiguousarray(np.array(nu_p, np.int32)),
                A=A, b=b, Ea=Ea)


def _trig_field(X, L, seed, stream, nmodes=4):
    """smooth periodic field with values in [-1,1]: normalised sum of low trig modes"""
    dim = X.shape[1]
    r = uniform(seed, stream, np.arange(nmodes * (dim + 2))).reshape(nmodes, dim + 2)
    acc = np.zeros_like(X[:, 0, :])
    tot = 0.0
    for m in range(nmodes):
        kvec = np.floor(r[m, :dim] * 3.0).astype(int)  # wave numbers 0..2
        if not kvec.any():
            kvec[m % dim] = 1
        amp = 0.5 + r[m, dim]
        ph = 2.0 * math.pi * r[m, dim + 1]
        arg = ph
        for c in range(dim):
            arg = arg + 2.0 * math.pi * kvec[c] * X[:, c, :] / L
        acc = acc + amp * np.sin(arg)
        tot += amp
    return acc / tot


def reacting_field(mesh: Mesh, L, seed=SEED):
    """config 5: T in [2000,9000] K, p in [1e3,1e5] Pa, |u_c| <= 500 m/s, Y = smooth
    partition-of-unity blend of 8 seeded Dirichlet(1,..,1) anchor compositions."""
    k = mesh.mech
    X = mesh.node_xyz
    T = 5500.0 + 3500.0 * _trig_field(X, L, seed, 61)
    p = 10.0 ** (4.0 + _trig_field(X, L, seed, 62))
    vel = [500.0 * _trig_field(X, L, seed, 63 + c) for c in range(mesh.dim)]
    na = 8
    g = -np.log(1.0 - uniform(seed, 71, np.arange(na * k.ns)).reshape(na, k.ns))  # Exp(1) draws
    anchors = g / g.sum(axis=1, keepdims=True)  # Dirichlet(1,...,1)
    wts = [(1.0 + _trig_field(X, L, seed, 80 + a)) ** 2 + 0.1 for a in range(na)]
    wsum = sum(wts)
    Y = [sum(wts[a] * anchors[a, s] for a in range(na)) / wsum for s in range(k.ns)]
    Rmix = sum(Y[s] * R_UNIVERSAL / k.W[s] for s in range(k.ns))
    rho = p / (Rmix * T)
    e = np.zeros_like(T)
    for s in range(k.ns):
        a = np.where((T < k.T_mid)[..., None], k.nasa[s, 0], k.nasa[s, 1])
        h_RT = (a[..., 0] + a[..., 1] * T / 2 + a[..., 2] * T ** 2 / 3 + a[..., 3] * T ** 3 / 4
                + a[..., 4] * T ** 4 / 5 + a[..., 5] / T)
        e = e + Y[s] * (R_UNIVERSAL / k.W[s]) * T * (h_RT - 1.0)
    E = rho * e + 0.5 * rho * sum(v * v for v in vel)
    return np.ascontiguousarray(np.stack([rho * Y[s] for s in range(k.ns)] + [rho * v for v in vel] + [E], axis=1))


# ----------------------------------------------------------------------------
# the five configs of BASELINE.json (scale < 1 gives the small parity instances)
# ----------------------------------------------------------------------------
@dataclass
class Case:
    name: str
    mesh: Mesh
    u0: np.ndarray
    steps: int
    cfl: float = 0.5


C5_LENGTH = 2.0e-7  # metres (domain edge of the 32^3 instance); chosen per DESIGN.md section 5 (explicit-chemistry step <= 0.05 x fastest depletion time)


def make_case(name: str, cells=None, steps=None, order="morton") -> Case:
    """name in c1..c5 (c4 = the mortar-dense band instance, c4w = the ~250K-element wide one).
    `cells` overrides the elements per direction (base grid for c4) to get small instances."""
    if name == "c1":
        k = cells or 16
        m = cartesian_mesh(2, 3, (k, k), (0.0, 0.0), (10.0, 10.0), order=order)
        return Case(name, m, isentropic_vortex(m), steps or 100)
    if name == "c2":
        k = cells or 32
        m = cartesian_mesh(3, 4, (k,) * 3, (0.0,) * 3, (2 * math.pi,) * 3, order=order)
        # CFL 0.4: eq. 18 has no dimension factor and 0.5 is linearly unstable for SSP-RK33 at N=4 in 3-D (R11b)
        return Case(name, m, taylor_green(m, noise=1e-3), steps or 20, cfl=0.4)
    if name == "c3":
        k = cells or 64
        lo, hi = (0.0,) * 3, (2 * math.pi,) * 3
        m = cartesian_mesh(3, 3, (k,) * 3, lo, hi, order=order, warp=sine_warp((k,) * 3, lo, hi, k=min(8, max(1, k // 2))))
        m.physics, m.mu, m.Pr = NAVIER_STOKES, 1.0 / 1600.0, 0.72
        return Case(name, m, taylor_green(m), steps or 10)
    if name in ("c4", "c4w"):
        base = (cells, max(1, cells // 4)) if cells else (128, 32)
        wide = name == "c4w"
        m = quadtree_mesh(3, base=base, band=2.8 if wide else 0.15, jitter=0.0 if wide else 0.3)
        m.bc_state = shock_states(m.gamma)
        return Case(name, m, mach10_shock(m, half_width=6.0 * m.info["h_fine"]), steps or 20)
    if name == "c5":
        k = cells or 32
        L = C5_LENGTH * k / 32.0  # small instances keep the element size (and so dt / tau_chem) of the 32^3 one
        m = cartesian_mesh(3, 3, (k,) * 3, (0.0,) * 3, (L,) * 3, order=order)
        m.physics, m.mech = REACTING_EULER, air5_mechanism()
        return Case(name, m, reacting_field(m, L), steps or 10)
    raise ValueError(name)
