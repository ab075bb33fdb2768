"""Honest CPU blocking: renormalized operators of a left or right block.

Problem setup for cfg 1-2 and the tiny truncated pins (BASELINE.json: "operators
are built by CPU blocking with seeded random quantum-number-preserving orthonormal
isometries").  Renormalization is Eq. (8): O_new = W^T O_enlarged W,
W sector-block-diagonal with orthonormal columns.  The enlarged operators follow
the bipartition identities of DESIGN.md (readings 2, 6) with explicit
Jordan-Wigner factors Z = (-1)^N of the left factor:

  a+_p   : p in l: a+ x 1                      p in r: Z x a+
  A_pq   : (l,l) A x 1; (r,r) 1 x A;           (p in l, q in r): (a+_p Z) x a+_q
  B_pt   : (l,l) B x 1; (r,r) 1 x B;           (p in l, t in r): (a+_p Z) x a_t
  H'     = H x 1 + 1 x H + sum_{p in l}[(a+_p Z) x S_p + h.c.]
           + sum_{p in r}[-(S_p Z) x a+_p + h.c.]
           + [compl. P of the block x A of the site + h.c.] + sum Q(block) x B(site)
  S_p'   = S_p x 1 + Z x S_p + sum_{q in l} a+_q x P_pq + sum_{q in r} (P_pq Z) x a+_q
           + sum_{t in l} a_t x Q_pt + sum_{r in r} (Q_pr Z) x a_r

One of the two factors is always a single site; the block's complementary
operators are formed from its carried A, B by  P_pq = sum_{s<r} V[p,q,s,r] A_sr^T,
Q_ps = sum_{q,r} V[p,q,s,r] B_qr  (definitions).  Products inside a
block are carried as their own renormalized operators, never recomposed.

Every "transpose" below is the Hermitian conjugate (a_p = (a+_p)^H): the plain transpose for the real
spin-free integrals, the conjugate transpose for the complex integrals of a spin-orbit Hamiltonian
(PAPER.md:97), for which the bases carry N only (ints.sym == "N"), the isometries are complex and a
single site has the three sectors N = 0, 1, 2 of dimensions 1, 2, 1.
"""
import numpy as np

from .conventions import site_q
from .sectors import full_dim, kept_dims
from .siteops import SiteOps


class RBlock:
    """A (renormalized) block: sector table + block-sparse operators.

    ops[key] = {(row_sector, col_sector): ndarray}, keys ('C',p) ('A',p,q) p<q
    ('B',p,t) p<=t ('S',p) ('H',)."""

    def __init__(self, labels, sectors, dims):
        self.labels = list(labels)
        self.sectors = list(sectors)
        self.dims = list(dims)
        self.index = {q: i for i, q in enumerate(self.sectors)}
        self.ops = {}

    @property
    def norb(self):
        return len(self.labels) // 2

    # ---- derived operators (block-sparse dicts) ------------------------
    def transpose(self, blocks):
        return {(c, r): m.conj().T for (r, c), m in blocks.items()}

    def Bfull(self, p, t):
        return self.ops[("B", p, t)] if p <= t else self.transpose(self.ops[("B", t, p)])

    def compl_P(self, p, q, ints):
        """P_pq = sum_{s<r in X} V[p,q,s,r] a_r a_s = sum V (A_sr)^T."""
        out = {}
        X = self.labels
        for i, s in enumerate(X):
            for r in X[i + 1:]:
                v = ints.V(p, q, s, r)
                if v != 0.0:
                    for (rr, cc), m in self.ops[("A", s, r)].items():
                        _acc(out, (cc, rr), v * m.conj().T)
        return out

    def compl_Q(self, p, s, ints):
        """Q_ps = sum_{q,r in X} V[p,q,s,r] a+_q a_r."""
        out = {}
        X = self.labels
        for q in X:
            for r in X:
                v = ints.V(p, q, s, r)
                if v != 0.0:
                    for key, m in self.Bfull(q, r).items():
                        _acc(out, key, v * m)
        return out


def _acc(d, key, m):
    if key in d:
        d[key] = d[key] + m
    else:
        d[key] = m.copy() if isinstance(m, np.ndarray) else m


def site_block(k, ints, outside):
    """Exact single-site block with all carried operators (S_p for p in `outside`)."""
    so = SiteOps(k, ints)
    sym = getattr(ints, "sym", "NSz")
    a, b = so.labels
    if sym == "NSz":
        where = [(0, 0), (1, 0), (2, 0), (3, 0)]          # site state -> (sector, position inside it)
        blk = RBlock(so.labels, list(site_q(sym)), [1, 1, 1, 1])
        blk.dets = {0: [0], 1: [1 << b], 2: [1 << a], 3: [(1 << a) | (1 << b)]}
    else:
        where = [(0, 0), (1, 0), (1, 1), (2, 0)]
        blk = RBlock(so.labels, [(0, 0), (1, 0), (2, 0)], [1, 2, 1])
        blk.dets = {0: [0], 1: [1 << b, 1 << a], 2: [(1 << a) | (1 << b)]}

    def sparse(m):
        out = {}
        for i in range(4):
            for j in range(4):
                if m[i, j] != 0.0:
                    (si, pi), (sj, pj) = where[i], where[j]
                    if (si, sj) not in out:
                        out[(si, sj)] = np.zeros((blk.dims[si], blk.dims[sj]), dtype=np.asarray(m).dtype)
                    out[(si, sj)][pi, pj] = m[i, j]
        return out

    for p in so.labels:
        blk.ops[("C", p)] = sparse(so.C(p))
    blk.ops[("A", a, b)] = sparse(so.A(a, b))
    for p in so.labels:
        for t in so.labels:
            if p <= t:
                blk.ops[("B", p, t)] = sparse(so.B(p, t))
    for p in outside:
        blk.ops[("S", p)] = sparse(so.S(p))
    blk.ops[("H",)] = sparse(so.H())
    # determinant bookkeeping (tiny-K pins): the site states of each sector, one determinant each
    blk.E = {i: np.eye(d) for i, d in enumerate(blk.dims)}
    return blk


def _zr(blocks, blk):
    """O Z: scale column sector q by (-1)^N(q)."""
    return {(r, c): (m if blk.sectors[c][0] % 2 == 0 else -m) for (r, c), m in blocks.items()}


def _ident(blk):
    return {(i, i): np.eye(d) for i, d in enumerate(blk.dims)}


def _zdiag(blk):
    return {(i, i): np.eye(d) * (-1.0) ** blk.sectors[i][0] for i, d in enumerate(blk.dims)}


class _Enlarged:
    """Product basis |l>|r>, grouped into sectors q' = q_l + q_r (left-major Kronecker)."""

    def __init__(self, left, right):
        self.left, self.right = left, right
        sub = {}
        for il, ql in enumerate(left.sectors):
            for ir, qr in enumerate(right.sectors):
                q = (ql[0] + qr[0], ql[1] + qr[1])
                sub.setdefault(q, []).append((il, ir))
        self.sectors = sorted(sub)
        self.index = {q: i for i, q in enumerate(self.sectors)}
        self.offset = {}
        self.dims = []
        for i, q in enumerate(self.sectors):
            off = 0
            for il, ir in sub[q]:
                self.offset[(il, ir)] = (i, off)
                off += left.dims[il] * right.dims[ir]
            self.dims.append(off)

    def kron_add(self, out, Ol, Or, coef=1.0):
        """out += coef * (Ol x Or), both block-sparse dicts."""
        for (rl, cl), ml in Ol.items():
            for (rr, cr), mr in Or.items():
                (a, ro) = self.offset[(rl, rr)]
                (b, co) = self.offset[(cl, cr)]
                k = np.kron(ml, mr) * coef
                if (a, b) not in out:
                    out[(a, b)] = np.zeros((self.dims[a], self.dims[b]), dtype=k.dtype)
                elif out[(a, b)].dtype != k.dtype and k.dtype.kind == "c":
                    out[(a, b)] = out[(a, b)].astype(k.dtype)
                out[(a, b)][ro:ro + k.shape[0], co:co + k.shape[1]] += k


def merge(left, right, ints, outside, K, N_tot, twoSz_tot, D, rng=None, rotate=False,
          force_dmax=True, site_side=None, track=False):
    """Enlarge: new block = left x right (one of them a single site), then renormalize.

    outside: labels p for which S_p of the NEW block is carried.
    D: max kept states (None = keep everything that can reach the target).
    rng: numpy Generator for the isometries; rotate=True applies a random orthogonal
    rotation even when nothing is truncated."""
    assert left.norb == 1 or right.norb == 1
    sym = getattr(ints, "sym", "NSz")
    cplx = np.dtype(getattr(ints, "dtype", np.float64)).kind == "c"
    if site_side is None:
        site_side = "right" if right.norb == 1 else "left"
    site_is_right = site_side == "right"
    blk, site = (left, right) if site_is_right else (right, left)
    assert site.norb == 1
    E = _Enlarged(left, right)
    Il, Ir = _ident(left), _ident(right)
    Zl = _zdiag(left)
    T = left.transpose
    ops = {}

    def prod(Ol, Or, coef=1.0, into=None):
        out = {} if into is None else into
        E.kron_add(out, Ol, Or, coef)
        return out

    labs_l, labs_r = left.labels, right.labels
    # a+_p
    for p in labs_l:
        ops[("C", p)] = prod(left.ops[("C", p)], Ir)
    for p in labs_r:
        ops[("C", p)] = prod(Zl, right.ops[("C", p)])
    # A_pq, B_pt
    CZ = {p: _zr(left.ops[("C", p)], left) for p in labs_l}            # a+_p Z
    DZ = {p: _zr(T(left.ops[("C", p)]), left) for p in labs_l}         # a_p Z
    Dr = {p: right.transpose(right.ops[("C", p)]) for p in labs_r}     # a_p on the right factor
    for i, p in enumerate(labs_l):
        for q in labs_l[i + 1:]:
            ops[("A", p, q)] = prod(left.ops[("A", p, q)], Ir)
        for t in labs_l[i:]:
            ops[("B", p, t)] = prod(left.ops[("B", p, t)], Ir)
        for q in labs_r:
            ops[("A", p, q)] = prod(CZ[p], right.ops[("C", q)])
            ops[("B", p, q)] = prod(CZ[p], Dr[q])
    for i, p in enumerate(labs_r):
        for q in labs_r[i + 1:]:
            ops[("A", p, q)] = prod(Il, right.ops[("A", p, q)])
        for t in labs_r[i:]:
            ops[("B", p, t)] = prod(Il, right.ops[("B", p, t)])
    # H'
    Hn = prod(left.ops[("H",)], Ir)
    prod(Il, right.ops[("H",)], into=Hn)
    for p in labs_l:   # (a+_p Z) x S_p^r + h.c.
        Sr = right.ops[("S", p)]
        prod(CZ[p], Sr, into=Hn)
        prod(T(CZ[p]), right.transpose(Sr), into=Hn)
    for p in labs_r:   # -(S_p^l Z) x a+_p + h.c.
        SZ = _zr(left.ops[("S", p)], left)
        prod(SZ, right.ops[("C", p)], -1.0, into=Hn)
        prod(T(SZ), Dr[p], -1.0, into=Hn)
    s0, s1 = site.labels
    Pb = blk.compl_P(s0, s1, ints)
    As = site.ops[("A", s0, s1)]
    if site_is_right:
        prod(Pb, As, into=Hn)
        prod(T(Pb), site.transpose(As), into=Hn)
        for p in site.labels:
            for t in site.labels:
                prod(blk.compl_Q(p, t, ints), site.Bfull(p, t), into=Hn)
    else:
        prod(As, Pb, into=Hn)
        prod(site.transpose(As), blk.transpose(Pb), into=Hn)
        for p in site.labels:
            for t in site.labels:
                prod(site.Bfull(p, t), blk.compl_Q(p, t, ints), into=Hn)
    ops[("H",)] = Hn
    # S_p'
    for p in outside:
        Sn = prod(left.ops[("S", p)], Ir)
        prod(Zl, right.ops[("S", p)], into=Sn)
        for q in labs_l:    # a+_q x P^r_pq ; a_q x Q^r_pq
            prod(left.ops[("C", q)], right.compl_P(p, q, ints), into=Sn)
            prod(T(left.ops[("C", q)]), right.compl_Q(p, q, ints), into=Sn)
        for q in labs_r:    # (P^l_pq Z) x a+_q ; (Q^l_pq Z) x a_q
            prod(_zr(left.compl_P(p, q, ints), left), right.ops[("C", q)], into=Sn)
            prod(_zr(left.compl_Q(p, q, ints), left), Dr[q], into=Sn)
        ops[("S", p)] = Sn
    # ---- renormalize -----------------------------------------------------
    m_new = left.norb + right.norb
    if D is None:
        rest = K - m_new
        keep = [d if full_dim(rest, N_tot - q[0], twoSz_tot - q[1], sym) > 0 else 0
                for q, d in zip(E.sectors, E.dims)]
    else:
        keep = list(kept_dims(E.sectors, E.dims, m_new, K, N_tot, twoSz_tot, D, force_dmax, sym))
    W = {}
    new_secs, new_dims, remap = [], [], {}
    for i, (q, d, k) in enumerate(zip(E.sectors, E.dims, keep)):
        k = int(k)
        if k <= 0:
            continue
        if k == d and not rotate:
            W[i] = None
        else:
            g = rng.standard_normal((d, d))
            if cplx:
                g = g + 1j * rng.standard_normal((d, d))
            qmat, _ = np.linalg.qr(g)
            W[i] = qmat[:, :k]
        remap[i] = len(new_secs)
        new_secs.append(q)
        new_dims.append(k)
    nb = RBlock(labs_l + labs_r, new_secs, new_dims)
    # the site tensor A of Eq. (8) as the renormalization step consumes it: one sub-block per
    # (old-block sector, site state) -> new sector, rows of the kept isometry W (identity where nothing is rotated)
    nb.site_tensor = []
    for (il, ir), (a, off) in sorted(E.offset.items()):
        if a not in remap or sym != "NSz":   # (the renormalization step is built for the N, Sz bases only)
            continue
        d = left.dims[il] * right.dims[ir]
        Wa = np.eye(E.dims[a]) if W[a] is None else W[a]
        i_old, n_site = (il, ir) if site_is_right else (ir, il)
        nb.site_tensor.append((i_old, n_site, remap[a], np.ascontiguousarray(Wa[off:off + d, :])))
    for key, blocks in ops.items():
        out = {}
        for (a, b), m in blocks.items():
            if a not in remap or b not in remap:
                continue
            x = m if W[a] is None else W[a].conj().T @ m
            x = x if W[b] is None else x @ W[b]
            out[(remap[a], remap[b])] = x
        nb.ops[key] = out
    nb.dets, nb.E = None, None
    if track and getattr(left, "dets", None) is not None and getattr(right, "dets", None) is not None:
        # isometry from the determinant basis: E_new = blockdiag(kron(E_l, E_r)) W   (tiny K only)
        nb.dets, nb.E = {}, {}
        sub = {}
        for (il, ir), (a, off) in E.offset.items():
            sub.setdefault(a, []).append((off, il, ir))
        for a, lst in sub.items():
            if a not in remap:
                continue
            dets, mats = [], []
            for off, il, ir in sorted(lst):
                dets += [dl | dr for dl in left.dets[il] for dr in right.dets[ir]]
                mats.append(np.kron(left.E[il], right.E[ir]))
            nr = sum(m.shape[0] for m in mats)
            Ee = np.zeros((nr, E.dims[a]), dtype=np.result_type(*[m.dtype for m in mats]))
            r0 = c0 = 0
            for m in mats:
                Ee[r0:r0 + m.shape[0], c0:c0 + m.shape[1]] = m
                r0 += m.shape[0]
                c0 += m.shape[1]
            nb.dets[remap[a]] = dets
            nb.E[remap[a]] = Ee if W[a] is None else Ee @ W[a]
    return nb


def build_block(side, sites, ints, K, N_tot, twoSz_tot, D, rng=None, rotate=False,
                force_dmax=True, track=False):
    """Grow a block over `sites` (list of spatial orbitals).  side 'L': sites ascending,
    new site appended on the right; side 'R': sites descending, new site on the left."""
    order = list(sites) if side == "L" else list(sites)[::-1]
    inside = []
    blk = None
    for k in order:
        inside.append(k)
        outside = [P for P in range(2 * K) if (P >> 1) not in inside]
        site = site_block(k, ints, [P for P in range(2 * K) if (P >> 1) != k])
        if blk is None:
            blk = site
            continue
        if side == "L":
            blk = merge(blk, site, ints, outside, K, N_tot, twoSz_tot, D, rng, rotate, force_dmax,
                        site_side="right", track=track)
        else:
            blk = merge(site, blk, ints, outside, K, N_tot, twoSz_tot, D, rng, rotate, force_dmax,
                        site_side="left", track=track)
    return blk
