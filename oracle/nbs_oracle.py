"""CPU oracle for the HAL QCD four-point function F(r) of arXiv:1604.07983.

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
`cpu_baseline` / `--impl reference` legs may import this module.  It shares no code with the CUDA
path (`paper_1604_07983_b200/`), and the CUDA path never imports it.  Plain numpy, fp64/complex128.

Three tiers, each pinned by the one before (tests/test_oracle_*.py):

  tier W  `oracle/wick.c`           brute-force Wick contraction of the interpolating operators
                                    of eqs. 2.2-2.3 (6x6 determinant per index tuple).
  tier A  `correlator_direct`       eq. 2.4 written out: normal baryon blocks (eq. 2.5), the sum
                                    over permutations P with sigma_P, the eps.eps.Cg5.Cg5.d.d
                                    weights, and the direct sum over X.  O(V^2).
  tier B  `correlator_fft`          eq. 2.6 / section 4 in the paper's order: (i) normal blocks,
                                    FFT; (ii) effective blocks per diagram (eq. 4.2); (iii) their
                                    product summed over the shared index (eq. 4.3), summed over
                                    diagrams with sigma_P; inverse FFT.

Conventions (readings A1-A17 of DESIGN.md):
  xi = colour + 3*spin (12 values); propagator S_f[x][sink xi][source xi']; site x + L*(y + L*z);
  C gamma_5 = [[0,1,0,0],[-1,0,0,0],[0,0,0,1],[0,0,-1,0]]  (Dirac basis, C = gamma_4 gamma_2);
  periodic space; F(r) = sum_X <B1(X+r) B2(X) Jbar>; output F[a1][a2][a3][a4][r].

Parity status: every function here is pinned (tier W, closed forms, the paper's printed counts,
symmetry relations) EXCEPT absolute values of F on the paper's own lattices, which the paper
never prints -> those are "parity unpinned against the paper" (oracle <-> CUDA only).
"""
from __future__ import annotations

import itertools
import math

import numpy as np
import scipy.sparse as sp

NC, NA, NX = 3, 4, 12

# ---------------------------------------------------------------------------------------------
# Constant tensors (eqs. 2.2-2.3; eq. 2.4)
# ---------------------------------------------------------------------------------------------
EPS = np.zeros((3, 3, 3))
for _p in itertools.permutations(range(3)):
    _inv = sum(1 for i in range(3) for j in range(i + 1, 3) if _p[i] > _p[j])
    EPS[_p] = -1.0 if _inv % 2 else 1.0

# Reading A1: the paper never states its gamma basis.
CG5 = np.array([[0, 1, 0, 0], [-1, 0, 0, 0], [0, 0, 0, 1], [0, 0, -1, 0]], dtype=float)


def _build_W() -> np.ndarray:
    """W[xi1, xi2, xi3; a] = eps_{c1 c2 c3} (C g5)_{a1 a2} delta_{a3 a}: the colour-spin weight of
    every elementary operator eps_abc (q1_a C g5 q2_b) q3_c (eq. 2.2-2.3), and of the source
    factors eps eps Cg5 Cg5 delta delta in eq. 2.4."""
    W = np.zeros((NX, NX, NX, NA))
    for c1, c2, c3 in itertools.product(range(3), repeat=3):
        for a1, a2, a in itertools.product(range(4), repeat=3):
            W[c1 + 3 * a1, c2 + 3 * a2, c3 + 3 * a, a] = EPS[c1, c2, c3] * CG5[a1, a2]
    return W


W = _build_W()

_S6, _S2 = 1.0 / math.sqrt(6.0), 1.0 / math.sqrt(2.0)

# name -> (slot flavours g1g2g3 of the block, eq. 2.5; elementary terms (coefficient, f1f2f3) with
# E[f1f2f3] = eps_abc (f1_a C g5 f2_b) f3_c).  Eqs. 2.2 and 2.3 verbatim.
BARYONS: dict[str, tuple[str, list[tuple[float, str]]]] = {
    "p": ("udu", [(+1.0, "udu")]),
    "n": ("udd", [(-1.0, "udd")]),
    "Sp": ("usu", [(-1.0, "usu")]),
    "Sm": ("dsd", [(-1.0, "dsd")]),
    "X0": ("uss", [(+1.0, "uss")]),
    "Xm": ("dss", [(-1.0, "dss")]),
    "Xu": ("uds", [(1.0, "dsu")]),
    "Xd": ("uds", [(1.0, "sud")]),
    "Xs": ("uds", [(1.0, "uds")]),
    "L": ("uds", [(_S6, "dsu"), (_S6, "sud"), (-2.0 * _S6, "uds")]),
    "S0": ("uds", [(_S2, "dsu"), (-_S2, "sud")]),
}

# Reading A10: the 52 channels "from NN to Xi-Xi"; the list itself is in Ref. [14]
# which is not available.  Sectors of fixed strangeness and charge; all sink x source pairs inside a
# sector except the four isospin-forbidden ones.
SECTORS = [
    [("p", "n")],
    [("p", "L"), ("Sp", "n"), ("S0", "p")],
    [("L", "L"), ("p", "Xm"), ("n", "X0"), ("Sp", "Sm"), ("S0", "S0"), ("S0", "L")],
    [("Xm", "L"), ("Sm", "X0"), ("S0", "Xm")],
    [("Xm", "X0")],
]
_FORBIDDEN = {(("L", "L"), ("S0", "L")), (("S0", "L"), ("L", "L")),
              (("S0", "S0"), ("S0", "L")), (("S0", "L"), ("S0", "S0"))}


def channels52() -> list[tuple[str, str, str, str]]:
    out = []
    for sec in SECTORS:
        for snk in sec:
            for src in sec:
                if (snk, src) in _FORBIDDEN:
                    continue
                out.append((snk[0], snk[1], src[0], src[1]))
    return out


# ---------------------------------------------------------------------------------------------
# Permutations P and signs sigma_P (eq. 2.4)
# ---------------------------------------------------------------------------------------------
def perm_sign(P) -> int:
    inv = sum(1 for i in range(len(P)) for j in range(i + 1, len(P)) if P[i] > P[j])
    return -1 if inv % 2 else 1


def slot_multiplicity(name: str) -> int:
    """m = prod_flavours (number of slots of that flavour)!  (2 for p,n,Sigma+-,Xi; 1 otherwise)."""
    g = BARYONS[name][0]
    return math.prod(math.factorial(g.count(f)) for f in "uds")


def _is_coset_rep(P, g) -> bool:
    for base in (0, 3):
        for j in range(base, base + 3):
            for k in range(j + 1, base + 3):
                if g[j] == g[k] and P[j] > P[k]:
                    return False
    return True


def diagrams(ch, all_perms: bool = False):
    """All terms of eq. 2.4 for channel ch = (B1, B2, B3, B4): a list of (coef, sigma_P, P) with
    P[j] = index (0..5) of the source quark sitting in sink slot j (slots 0-2 of B1, 3-5 of B2);
    source quarks 0-2 belong to B3, 3-5 to B4, numbered in the elementary operator's field order.
    Source Lambda / Sigma0 are expanded into their X_u, X_d, X_s terms (coef = k3*k4, the same
    real coefficients as at the sink, reading A4).  By default one P per coset modulo exchange of
    same-flavour slots inside one sink baryon (reading A5: the block is antisymmetric under that
    exchange, which is the paper's factor 2^{N_Lambda+N_Sigma0-B}); all_perms=True returns every
    flavour-preserving P (to be divided by m1*m2)."""
    b1, b2, b3, b4 = ch
    g = BARYONS[b1][0] + BARYONS[b2][0]
    out = []
    for k3, h3 in BARYONS[b3][1]:
        for k4, h4 in BARYONS[b4][1]:
            h = h3 + h4
            for P in itertools.permutations(range(6)):
                if any(g[j] != h[P[j]] for j in range(6)):
                    continue
                if not all_perms and not _is_coset_rep(P, g):
                    continue
                out.append((k3 * k4, perm_sign(P), P))
    return out


def cut_positions(P, side: int, src: int) -> tuple[int, ...]:
    """Positions (1,2,3) of source baryon `src` (0: B3, 1: B4) whose quarks sit in sink `side`."""
    return tuple(sorted(q % 3 + 1 for q in P[3 * side:3 * side + 3] if q // 3 == src))


def shared_size(A: tuple[int, ...]) -> int:
    """Size of the shared index when W is cut into positions A | complement:
    1 if nothing is cut, N_c if the C g5 pair {1,2} is split from quark 3, N_c N_alpha otherwise."""
    if len(A) in (0, 3):
        return 1
    if A in ((1, 2), (3,)):
        return NC
    return NC * NA


def diagram_K(P) -> int:
    return shared_size(cut_positions(P, 0, 0)) * shared_size(cut_positions(P, 0, 1))


# ---------------------------------------------------------------------------------------------
# (i) Normal baryon blocks, eq. 2.5 / 4.1
# ---------------------------------------------------------------------------------------------
def elementary_T(S: dict, f: str) -> np.ndarray:
    """T^{f1f2f3}[x, a, xi1, xi2, xi3] = sum_eta W[eta; a] S_f1[x, eta1, xi1] S_f2[x, eta2, xi2]
    S_f3[x, eta3, xi3]: the elementary operator with its three quarks propagated to source
    indices xi1, xi2, xi3 (field order), no exchange terms."""
    V = S[f[0]].shape[0]
    S1 = S[f[0]].reshape(V, 4, 3, NX)  # [x, spin, colour, source]
    S2 = S[f[1]].reshape(V, 4, 3, NX)
    S3 = S[f[2]].reshape(V, 4, 3, NX)
    D = np.einsum("abc,st,xsai,xtbj->xcij", EPS, CG5, S1, S2, optimize=True)
    return np.einsum("xcij,xsck->xsijk", D, S3, optimize=True)


def block(S: dict, name: str) -> np.ndarray:
    """[B_a](x; xi1, xi2, xi3) = <B_a(x) qbar_3(xi3) qbar_2(xi2) qbar_1(xi1)> with the source quarks
    in the slot-flavour order g of BARYONS[name]:  sum over elementary terms and over the Wick
    pairings sigma (field j -> slot sigma(j), same flavour) with sign sgn(sigma)."""
    g, terms = BARYONS[name]
    out = None
    for k, f in terms:
        T = elementary_T(S, f)
        for sig in itertools.permutations(range(3)):
            if any(f[j] != g[sig[j]] for j in range(3)):
                continue
            inv = [0, 0, 0]
            for j in range(3):
                inv[sig[j]] = j  # slot m is fed by field inv[m]
            term = k * perm_sign(sig) * np.transpose(T, (0, 1, 2 + inv[0], 2 + inv[1], 2 + inv[2]))
            out = term if out is None else out + term
    return np.ascontiguousarray(out)


# ---------------------------------------------------------------------------------------------
# Tier A: eq. 2.4 literally
# ---------------------------------------------------------------------------------------------
def _ww_nonzeros():
    """The 96 x 96 non-zero entries of W[xi'1 xi'2 xi'3; a3] * W[xi'4 xi'5 xi'6; a4], grouped by
    (a3, a4): returns xi [6][16][576] and val [16][576]."""
    nz = np.argwhere(W != 0)  # rows (xi1, xi2, xi3, a)
    vals = W[W != 0]
    per_a = [(nz[nz[:, 3] == a][:, :3], vals[nz[:, 3] == a]) for a in range(4)]
    xi = np.zeros((6, 16, 576), dtype=np.int64)
    val = np.zeros((16, 576))
    for a3 in range(4):
        for a4 in range(4):
            t3, v3 = per_a[a3]
            t4, v4 = per_a[a4]
            G = a3 * 4 + a4
            i3, i4 = np.meshgrid(np.arange(24), np.arange(24), indexing="ij")
            i3, i4 = i3.ravel(), i4.ravel()
            for m in range(3):
                xi[m, G] = t3[i3, m]
                xi[3 + m, G] = t4[i4, m]
            val[G] = v3[i3] * v4[i4]
    return xi, val


_WW_XI, _WW_VAL = _ww_nonzeros()


def pair_tensor(B1x: np.ndarray, B2y: np.ndarray, ch, all_perms: bool = False) -> np.ndarray:
    """sum_P sigma_P sum_{xi'} W W [B1_a1](x; xi'_P1 xi'_P2 xi'_P3) [B2_a2](y; xi'_P4 xi'_P5 xi'_P6)
    for a batch of site pairs: B1x, B2y of shape [n, 4, 12, 12, 12] -> [n, 4, 4, 4, 4]."""
    n = B1x.shape[0]
    b1 = B1x.reshape(n, 4, 1728)
    b2 = B2y.reshape(n, 4, 1728)
    out = np.zeros((n, 4, 4, 16), dtype=np.complex128)
    norm = 1.0
    if all_perms:
        norm = 1.0 / (slot_multiplicity(ch[0]) * slot_multiplicity(ch[1]))
    for coef, sgn, P in diagrams(ch, all_perms):
        t1 = (_WW_XI[P[0]] * 12 + _WW_XI[P[1]]) * 12 + _WW_XI[P[2]]  # [16, 576]
        t2 = (_WW_XI[P[3]] * 12 + _WW_XI[P[4]]) * 12 + _WW_XI[P[5]]
        g1 = b1[:, :, t1]  # [n, 4, 16, 576]
        g2 = b2[:, :, t2]
        out += (coef * sgn * norm) * np.einsum("xaGt,xbGt,Gt->xabG", g1, g2, _WW_VAL, optimize=True)
    return out.reshape(n, 4, 4, 4, 4)


def _shift_index(L: int, r: int) -> np.ndarray:
    """site index of X + r for every site X (periodic, reading A8)."""
    V = L ** 3
    X = np.arange(V)
    x, y, z = X % L, (X // L) % L, X // (L * L)
    rx, ry, rz = r % L, (r // L) % L, r // (L * L)
    return ((x + rx) % L) + L * (((y + ry) % L) + L * ((z + rz) % L))


def correlator_direct(L: int, blocks: dict, ch, all_perms: bool = False, rs=None) -> np.ndarray:
    """Tier A.  F[a1,a2,a3,a4,r] = sum_X pair_tensor(B1(X+r), B2(X)) (eq. 2.4, reading A9).
    `blocks[name]` = block(S, name) of shape [V,4,12,12,12].  rs: optional subset of r."""
    V = L ** 3
    rs = range(V) if rs is None else rs
    F = np.zeros((4, 4, 4, 4, V), dtype=np.complex128)
    B1, B2 = blocks[ch[0]], blocks[ch[1]]
    for r in rs:
        F[..., r] = pair_tensor(B1[_shift_index(L, r)], B2, ch, all_perms).sum(axis=0)
    return F


# ---------------------------------------------------------------------------------------------
# Tier B: effective blocks (eqs. 2.6, 4.2, 4.3)
# ---------------------------------------------------------------------------------------------
def _cut_factor(A: tuple[int, ...]) -> np.ndarray:
    """Factor of W that goes to the side holding source positions A, with axes
    (xi_p for p in A ..., shared index, carried spin (4 if 3 in A else 1)), such that
    W[xi1 xi2 xi3; a] = sum_shared factor(A) * factor(complement of A)."""
    if A == ():
        return np.ones((1, 1))
    if A == (1, 2, 3):
        return W.reshape(NX, NX, NX, 1, NA)
    if A == (1, 2):  # eps_{c1 c2 c} (Cg5)_{a1 a2}, open colour c of quark 3
        F = np.zeros((NX, NX, NC, 1))
        for c1, c2, c in itertools.product(range(3), repeat=3):
            for a1, a2 in itertools.product(range(4), repeat=2):
                F[c1 + 3 * a1, c2 + 3 * a2, c, 0] = EPS[c1, c2, c] * CG5[a1, a2]
        return F
    if A == (3,):  # quark 3 read at xi3 = (c, a3): carries the source spin a3
        F = np.zeros((NX, NC, NA))
        for c in range(3):
            for a in range(4):
                F[c + 3 * a, c, a] = 1.0
        return F
    if A == (1, 3):  # W with the partner index xi2 left open
        return np.ascontiguousarray(np.transpose(W, (0, 2, 1, 3)))
    if A == (2, 3):  # W with the partner index xi1 left open
        return np.ascontiguousarray(np.transpose(W, (1, 2, 0, 3)))
    if A in ((1,), (2,)):  # the lone Cg5 partner: read raw at the shared index
        return np.eye(NX).reshape(NX, NX, 1)
    raise ValueError(A)


def side_tensor(slots: tuple[int, int, int]) -> np.ndarray:
    """For one sink baryon whose slots hold source quarks `slots` (ids 0..5): the tensor
    G[xi_slot1, xi_slot2, xi_slot3; carry3, carry4; s3, s4] that turns its normal block into its
    effective block (eq. 4.2).  carry3/carry4 have size 4 when this side holds the third quark
    of B3/B4 (it then carries a3/a4), else 1; s3, s4 are the shared indices xi~_d."""
    letters = "ijk"
    ops, subs = [], []
    for src, (sh, ca) in enumerate((("p", "c"), ("q", "d"))):
        pos = sorted((q % 3 + 1, letters[m]) for m, q in enumerate(slots) if q // 3 == src)
        A = tuple(p for p, _ in pos)
        ops.append(_cut_factor(A))
        subs.append("".join(l for _, l in pos) + sh + ca)
    return np.einsum(f"{subs[0]},{subs[1]}->ijkcdpq", ops[0], ops[1])


_SIDE_CACHE: dict = {}


def _side_sparse(slots):
    if slots not in _SIDE_CACHE:
        G = side_tensor(slots)
        shape = G.shape[3:]
        _SIDE_CACHE[slots] = (sp.csr_matrix(G.reshape(1728, -1).T), shape)
    return _SIDE_CACHE[slots]


def effective_block(Bq: np.ndarray, slots) -> np.ndarray:
    """(ii) EffectiveBaryonBlocks, eq. 4.2: Bq [n, 4, 12,12,12] -> e[n, 4, carry3, carry4, K]."""
    Gs, (c3, c4, s3, s4) = _side_sparse(tuple(slots))
    n = Bq.shape[0]
    e = (Gs @ Bq.reshape(n * 4, 1728).T).T
    return e.reshape(n, 4, c3, c4, s3 * s4)


def fourpt_momentum(B1q: np.ndarray, B2mq: np.ndarray, ch, cache=None) -> np.ndarray:
    """(ii)+(iii) for a batch of momenta: B1q = B~1(q), B2mq = B~2(-q), both [n,4,12,12,12].
    Returns sum_P sigma_P ( B~1^(P)(q) x B~2^(P)(-q) )_{a3 a4} as [n, 4,4,4,4] (eqs. 2.6, 4.3)."""
    n = B1q.shape[0]
    out = np.zeros((n, 4, 4, 4, 4), dtype=np.complex128)
    cache = {} if cache is None else cache
    for coef, sgn, P in diagrams(ch):
        k1, k2 = (ch[0], 0, P[:3]), (ch[1], 1, P[3:])
        if k1 not in cache:
            cache[k1] = effective_block(B1q, P[:3])
        if k2 not in cache:
            cache[k2] = effective_block(B2mq, P[3:])
        e1, e2 = cache[k1], cache[k2]
        # exactly one side carries a3 and exactly one carries a4 (sizes 4 and 1)
        prod = np.einsum("xacdk,xbefk->xabcedf", e1, e2, optimize=True)
        out += (coef * sgn) * prod.reshape(n, 4, 4, 4, 4)
    return out


def fft_blocks(L: int, B: np.ndarray) -> np.ndarray:
    """B~(q) = sum_x B(x) exp(-i q.x), q = 2 pi n / L, same site ordering for n as for x."""
    V = L ** 3
    return np.fft.fftn(B.reshape(L, L, L, -1), axes=(0, 1, 2)).reshape((V,) + B.shape[1:])


def minus_q_index(L: int) -> np.ndarray:
    V = L ** 3
    q = np.arange(V)
    x, y, z = q % L, (q // L) % L, q // (L * L)
    return ((-x) % L) + L * (((-y) % L) + L * ((-z) % L))


def correlator_fft(L: int, blocks: dict, chans, chunk: int = 512) -> np.ndarray:
    """Tier B.  F[ch, a1,a2,a3,a4, r] for the listed channels via eq. 2.6."""
    V = L ** 3
    names = sorted({b for ch in chans for b in ch[:2]})
    Bq = {b: fft_blocks(L, blocks[b]) for b in names}
    mq = minus_q_index(L)
    Ft = np.zeros((len(chans), V, 4, 4, 4, 4), dtype=np.complex128)
    for lo in range(0, V, chunk):
        hi = min(V, lo + chunk)
        caches: dict = {}
        for ic, ch in enumerate(chans):
            cache = caches.setdefault((ch[0], ch[1]), {})
            Ft[ic, lo:hi] = fourpt_momentum(Bq[ch[0]][lo:hi], Bq[ch[1]][mq[lo:hi]], ch, cache)
    F = np.fft.ifftn(Ft.reshape(len(chans), L, L, L, 256), axes=(1, 2, 3)).reshape(len(chans), V, 256)
    return np.ascontiguousarray(np.transpose(F, (0, 2, 1))).reshape(len(chans), 4, 4, 4, 4, V)


def all_blocks(S: dict, names) -> dict:
    return {b: block(S, b) for b in sorted(set(names))}


def sink_names(chans) -> list[str]:
    return sorted({b for ch in chans for b in ch[:2]})


def diagram_signature(P):
    """Human-readable structure of one diagram, for comparison with eq. 2.7 / PAPER.md:108:
    (K, shared index labels in the paper's primed numbering, spins carried by B~1, by B~2)."""
    labels, carry = [], ([], [])
    for src in (0, 1):
        A = cut_positions(P, 0, src)
        base = 3 * src
        if A in ((1, 2), (3,)):
            labels.append(f"c{base + 3}'")
        elif A in ((1, 3), (2,)):
            labels.append(f"c{base + 2}'a{base + 2}'")
        elif A in ((2, 3), (1,)):
            labels.append(f"c{base + 1}'a{base + 1}'")
        carry[0 if 3 in A else 1].append(f"a{3 + src}")
    return diagram_K(P), tuple(labels), tuple(carry[0]), tuple(carry[1])
