"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage or identity it checks.  A plausible mistake anywhere in the oracle
(a dropped diagram, a wrong sigma_P, a transposed propagator index, a wrong C g5 entry, a wrong
FFT sign) fails at least one of them.
"""
import itertools
import math

import numpy as np
import pytest

from conftest import read_golden
from oracle import nbs_oracle as O
from paper_1604_07983_b200 import synth

GOLD = read_golden("paper_counts.txt")


def rand_props(L, seed=11, same=()):
    S = {}
    for i, f in enumerate("uds"):
        S[f] = synth.propagator(seed, i, 0, L, 0.1)
    for a, b in same:
        S[a] = S[b]
    return S


@pytest.fixture(scope="module")
def lat2():
    S = rand_props(2)
    names = set(O.BARYONS)
    return S, O.all_blocks(S, names)


# ------------------------------------------------------------------ printed counts
def test_channel_count_is_52():
    assert len(O.channels52()) == int(GOLD["n_channels"])
    assert len(set(O.channels52())) == 52


def test_iteration_count_formula_3456():
    """(N_c! N_a)^B x N_u! N_d! N_s! x 2^{N_L+N_S0-B} = 3456 for <p L pbar Xubar>:
    the number of (coset-representative permutations) x (non-zero source index tuples)."""
    ch = ("p", "L", "p", "Xu")
    nperm = len(O.diagrams(ch))
    nz_per_spin = int((O.W[..., 0] != 0).sum())  # N_c! N_alpha = 24
    assert nz_per_spin == 24
    assert nperm * nz_per_spin ** 2 == int(GOLD["literal_terms_pLpXu"])
    # and the formula itself: N_u=3, N_d=2, N_s=1, N_Lambda=1 (sink), B=2
    assert 24 ** 2 * math.factorial(3) * math.factorial(2) * math.factorial(1) * 2 ** (1 + 0 - 2) == 3456
    # all flavour-preserving P = cosets x m1 x m2
    assert len(O.diagrams(ch, all_perms=True)) == nperm * O.slot_multiplicity("p") * O.slot_multiplicity("L")


def test_effective_count_370_and_sizes():
    """1 + 9 + 144 + 144 + 36 + 36 = 370."""
    Ks = [O.diagram_K(P) for _, _, P in O.diagrams(("p", "L", "p", "Xu"))]
    assert sum(Ks) == int(GOLD["effective_terms_pLpXu"])
    assert sorted(Ks) == sorted(int(v) for v in GOLD["effective_sizes_pLpXu"].split())


def test_eq_2_7_terms():
    """PAPER.md:65 (eq. 2.7) and :108: sign, shared index set and which block carries a3 / a4 for
    each printed term; the sixth index set {c1'a1' c5'a5'} (term lost in extraction, reading A6)."""
    got = {}
    for _, sgn, P in O.diagrams(("p", "L", "p", "Xu")):
        K, labels, c1, c2 = O.diagram_signature(P)
        got[" ".join(labels)] = ("+" if sgn > 0 else "-", " ".join(c1), " ".join(c2))
    for key in ("eq27_term_none", "eq27_term_c3c6", "eq27_term_c2a2c4a4", "eq27_term_c1a1c6", "eq27_term_c3c5a5"):
        sign, shared, c1, c2 = [s.strip() for s in GOLD[key].split(";")]
        assert got[shared] == (sign, c1, c2), key
    sets = [s.strip().replace("none", "") for s in GOLD["eq27_sets"].split("/")]
    assert sorted(sets) == sorted(got)


def test_derived_totals():
    """SURVEY.md 8(c) derived totals (not printed in the paper): 655 diagrams, sum K = 43507."""
    chans = O.channels52()
    ds = [O.diagram_K(P) for ch in chans for _, _, P in O.diagrams(ch)]
    assert len(ds) == 655 and sum(ds) == 43507
    hist = {k: ds.count(k) for k in set(ds)}
    assert hist == {1: 91, 9: 76, 36: 255, 144: 233}


# ------------------------------------------------------------------ constant tensors
def test_cg5_properties():
    """C g5 is real antisymmetric with (Cg5)(Cg5)^T = 1 and (Cg5)^2 = -1 (any standard basis)."""
    G = O.CG5
    assert np.array_equal(G, -G.T)
    assert np.array_equal(G @ G.T, np.eye(4)) and np.array_equal(G @ G, -np.eye(4))
    # Dirac basis: C = g4 g2, g5 = g1 g2 g3 g4 (reading A1) reproduces the matrix
    s = [np.array([[0, 1], [1, 0]]), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]])]
    Z = np.zeros((2, 2))
    g = [np.block([[Z, -1j * sk], [1j * sk, Z]]) for sk in s]
    g4 = np.diag([1, 1, -1, -1]).astype(complex)
    g5 = g[0] @ g[1] @ g[2] @ g4
    C = g4 @ g[1]
    assert np.allclose(C @ g5, G)


def test_cut_factors_reconstruct_W():
    """eq. 4.2: W = sum_shared factor(A) factor(complement) for every way of cutting the source."""
    for A, B, sub in [((1, 2), (3,), "ijpc,kpd->ijkcd"), ((1, 3), (2,), "ikpc,jpd->ijkcd"),
                      ((2, 3), (1,), "jkpc,ipd->ijkcd")]:
        R = np.einsum(sub, O._cut_factor(A), O._cut_factor(B))
        assert np.array_equal(R.reshape(12, 12, 12, 4), O.W), A


# ------------------------------------------------------------------ blocks (eq. 2.5)
def test_block_closed_form_normalisations():
    """With S_f(x) = s_f(x) 1: sum_xi W[xi;a'] [b_a](xi) = c_b delta_{aa'} prod s  (golden: hand-derived)."""
    V = 3
    rng = np.random.default_rng(5)
    s = {f: rng.standard_normal(V) + 1j * rng.standard_normal(V) for f in "uds"}
    S = {f: s[f][:, None, None] * np.eye(12)[None] for f in "uds"}
    expect = dict(Xs=24, p=30, n=-30, Sp=-30, Sm=-30, X0=30, Xm=-30, L=-60 / math.sqrt(6), S0=0)
    for name, key in [("Xs", "block_norm_Xs"), ("p", "block_norm_p"), ("n", "block_norm_n"),
                      ("Sp", "block_norm_Sp"), ("Sm", "block_norm_Sm"), ("X0", "block_norm_X0"),
                      ("Xm", "block_norm_Xm"), ("S0", "block_norm_S0")]:
        assert expect[name] == float(GOLD[key])
    assert float(GOLD["block_norm_L_times_sqrt6"]) == -60
    for name, c in expect.items():
        g = O.BARYONS[name][0]
        B = O.block(S, name)
        got = np.einsum("ijkb,xaijk->xab", O.W, B)
        ref = c * np.eye(4)[None] * np.prod([s[f] for f in g], axis=0)[:, None, None]
        assert np.allclose(got, ref, atol=1e-12), name


def test_block_antisymmetry_same_flavour_slots(lat2):
    _, bl = lat2
    assert np.allclose(bl["p"], -np.transpose(bl["p"], (0, 1, 4, 3, 2)))    # slots 1,3 = u,u
    assert np.allclose(bl["n"], -np.transpose(bl["n"], (0, 1, 2, 4, 3)))    # slots 2,3 = d,d
    assert np.allclose(bl["X0"], -np.transpose(bl["X0"], (0, 1, 2, 4, 3)))  # slots 2,3 = s,s
    assert np.allclose(bl["Sm"], -np.transpose(bl["Sm"], (0, 1, 4, 3, 2)))


def test_block_is_linear_combination(lat2):
    _, bl = lat2
    assert np.allclose(bl["L"], (bl["Xu"] + bl["Xd"] - 2 * bl["Xs"]) / math.sqrt(6))
    assert np.allclose(bl["S0"], (bl["Xu"] - bl["Xd"]) / math.sqrt(2))


def test_block_from_explicit_loops():
    """eq. 2.5 for the proton at one site, written as explicit loops over the 24 non-zeros of W."""
    S = rand_props(1, seed=3)
    B = O.block(S, "p")[0]
    Su, Sd = S["u"][0], S["d"][0]
    rng = np.random.default_rng(0)
    for _ in range(20):
        a, x1, x2, x3 = rng.integers(4), rng.integers(12), rng.integers(12), rng.integers(12)
        acc = 0
        for c1, c2, c3 in itertools.permutations(range(3)):
            for a1, a2 in ((0, 1), (1, 0), (2, 3), (3, 2)):
                w = O.EPS[c1, c2, c3] * O.CG5[a1, a2]
                e1, e2, e3 = c1 + 3 * a1, c2 + 3 * a2, c3 + 3 * a
                # u(e1) d(e2) u(e3) with source slots (u:x1, d:x2, u:x3): direct minus exchange
                acc += w * (Su[e1, x1] * Sd[e2, x2] * Su[e3, x3] - Su[e1, x3] * Sd[e2, x2] * Su[e3, x1])
        assert abs(acc - B[a, x1, x2, x3]) < 1e-12 * max(1, abs(acc))


# ------------------------------------------------------------------ tiers against each other
def test_tierA_equals_tierB_all_52_on_2cubed(lat2):
    """eq. 2.4 (direct X-sum, no factorisation) == eq. 2.6 (FFT + effective blocks)."""
    _, bl = lat2
    chans = O.channels52()
    FB = O.correlator_fft(2, bl, chans)
    for ic, ch in enumerate(chans):
        rs = [0, 3, 6] if ic % 4 else list(range(8))
        FA = O.correlator_direct(2, bl, ch, rs=rs)
        assert abs(FA[..., rs] - FB[ic][..., rs]).max() <= 1e-13 * abs(FA).max(), ch


def test_all_perms_over_m1m2_equals_coset_reps(lat2):
    """Reading A5 / PAPER.md:57: summing every P and dividing by m1 m2 = one P per coset."""
    _, bl = lat2
    for ch in [("p", "n", "p", "n"), ("Sp", "Sm", "S0", "S0"), ("Xm", "X0", "Xm", "X0")]:
        F1 = O.correlator_direct(2, bl, ch, rs=[0, 5])
        F2 = O.correlator_direct(2, bl, ch, all_perms=True, rs=[0, 5])
        assert abs(F1 - F2).max() <= 1e-13 * abs(F1).max()


# ------------------------------------------------------------------ symmetry relations (tier B, 2^3)
def _F(L, S, chans):
    bl = O.all_blocks(S, O.sink_names(chans))
    return O.correlator_fft(L, bl, chans)


def _close(a, b, tol=1e-12):
    return abs(a - b).max() <= tol * max(abs(a).max(), abs(b).max(), 1e-300)


def test_isospin_relations_u_equals_d():
    """north_star: 'isospin relations when u=d (pp and nn agree)'; SURVEY 8(c) in-list relations."""
    S = rand_props(2, seed=21, same=[("d", "u")])
    F = _F(2, S, [("p", "p", "p", "p"), ("n", "n", "n", "n"), ("p", "L", "p", "L"), ("n", "L", "n", "L")])
    assert _close(F[0], F[1]) and _close(F[2], F[3])
    ch = O.channels52()
    F52 = _F(2, S, ch)
    assert _close(F52[16], F52[23]) and _close(F52[17], F52[22])
    assert _close(F52[11], -F52[12]) and _close(F52[15], -F52[21]) and _close(F52[19], -F52[25])
    assert _close(F52[20], F52[26]) and _close(F52[34], -F52[35]) and _close(F52[38], F52[39])
    assert _close(F52[18], np.swapaxes(F52[24], 2, 3))
    # the four isospin-forbidden transitions of reading A10 vanish when u=d ...
    forb = [("L", "L", "S0", "L"), ("S0", "L", "L", "L"), ("S0", "S0", "S0", "L"), ("S0", "L", "S0", "S0")]
    Ff = _F(2, S, forb)
    assert abs(Ff).max() <= 1e-12 * abs(F52[10]).max()
    # ... and do not when u != d
    Ff2 = _F(2, rand_props(2, seed=21), forb)
    assert abs(Ff2).max() > 1e-3 * abs(F52[10]).max()


def test_su3_relations_u_equals_d_equals_s():
    """north_star: 'SU(3)-flavour relations when u=d=s'."""
    S = rand_props(2, seed=22, same=[("d", "u"), ("s", "u")])
    F = _F(2, S, [("p", "p", "p", "p"), ("Sp", "Sp", "Sp", "Sp"), ("X0", "X0", "X0", "X0"),
                  ("p", "n", "p", "n"), ("Sp", "X0", "Sp", "X0")])
    assert _close(F[0], F[1]) and _close(F[0], F[2]) and _close(F[3], F[4])


def test_swap_antisymmetries():
    """Reading A11: exchanging the two source baryons / the two sink baryons (Fermi statistics)."""
    S = rand_props(2, seed=23)
    F = _F(2, S, [("p", "L", "Sp", "n"), ("p", "L", "n", "Sp"), ("L", "p", "Sp", "n")])
    assert _close(F[0], -np.swapaxes(F[1], 2, 3))
    mr = O.minus_q_index(2)  # r -> -r
    assert _close(F[0], -np.swapaxes(F[2], 0, 1)[..., mr])
    FLL = _F(2, S, [("L", "L", "p", "Xm")])[0]
    assert _close(FLL, -np.swapaxes(FLL, 0, 1)[..., mr])


def test_flavour_scaling_and_linearity():
    S = rand_props(2, seed=24)
    chans = [("p", "L", "S0", "p"), ("p", "Xu", "S0", "p"), ("p", "Xd", "S0", "p"), ("p", "Xs", "S0", "p")]
    F = _F(2, S, chans)
    assert _close(F[0], (F[1] + F[2] - 2 * F[3]) / math.sqrt(6))
    lam = dict(u=1.3, d=0.7 + 0.2j, s=-0.4j)
    S2 = {f: lam[f] * S[f] for f in "uds"}
    F2 = _F(2, S2, chans[:1])
    assert _close(F2[0], lam["u"] ** 3 * lam["d"] ** 2 * lam["s"] * F[0])  # p L = uud uds


def test_local_colour_invariance():
    """eps_abc is an SU(3) invariant: S(x) -> U(x) S(x) V^+ with U(x) per site, V global."""
    L, V = 2, 8
    S = rand_props(L, seed=25)
    rng = np.random.default_rng(1)

    def su3():
        q, _ = np.linalg.qr(rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3)))
        return q / np.linalg.det(q) ** (1 / 3)

    U = np.stack([np.kron(np.eye(4), su3()) for _ in range(V)])  # xi = c + 3a: colour fastest
    Vg = np.kron(np.eye(4), su3())
    S2 = {f: U @ S[f] @ Vg.conj().T for f in "uds"}
    chans = [("p", "n", "p", "n"), ("S0", "L", "Sp", "Sm")]
    assert _close(_F(L, S, chans), _F(L, S2, chans), 1e-11)


def test_translation_delta_constant_and_tiling():
    """Textbook properties of the cyclic cross-correlation F(r) = sum_X B1(X+r) B2(X)."""
    L, V = 2, 8
    chans = [("p", "n", "p", "n"), ("p", "L", "Sp", "n")]
    S = rand_props(L, seed=26)
    F0 = _F(L, S, chans)
    sh = O._shift_index(L, 1 + 2 * 1)  # translate every propagator by (1,1,0)
    assert _close(F0, _F(L, {f: S[f][sh] for f in "uds"}, chans))
    # constant-in-x propagators: F(r) = V * G, independent of r
    Sc = {f: np.repeat(S[f][:1], V, axis=0) for f in "uds"}
    Fc = _F(L, Sc, chans)
    assert _close(Fc, np.repeat(Fc[..., :1], V, axis=-1))
    G = _F(1, {f: S[f][:1] for f in "uds"}, chans)
    assert _close(Fc[..., :1], V * G)
    # support on a single site x0: F(r) = delta_{r,0} G(x0,x0)
    Sd = {f: np.zeros_like(S[f]) for f in "uds"}
    for f in "uds":
        Sd[f][3] = S[f][0]
    Fd = _F(L, Sd, chans)
    assert _close(Fd[..., :1], G) and abs(Fd[..., 1:]).max() <= 1e-13 * abs(G).max()
    # tiling: a 4^3 field that repeats a 2^3 field 2x2x2 times gives 8 F_2(r mod 2)
    idx4 = np.arange(64)
    x, y, z = idx4 % 4, (idx4 // 4) % 4, idx4 // 16
    small = (x % 2) + 2 * ((y % 2) + 2 * (z % 2))
    F4 = _F(4, {f: S[f][small] for f in "uds"}, chans[:1])
    assert _close(F4[0], 8 * F0[0][..., small])


def test_pn_closed_form_with_diagonal_propagators():
    """With S_f = s_f(x) 1: F^{pn;pn}(r) = c d_{a1a3} d_{a2a4} sum_X (s_u^2 s_d)(X+r) (s_u s_d^2)(X);
    the constant c = 1080 is a pure combinatorial number, fixed here by the brute-force tier W on
    one site (not printed in the paper)."""
    from oracle import wick
    one = {f: np.eye(12, dtype=complex)[None] for f in "uds"}
    spins = [(0, 1, 0, 1), (2, 3, 2, 3), (0, 1, 1, 0), (0, 0, 0, 0), (1, 2, 1, 3)]
    c = wick.wick_fourpt(1, one, ("p", "n", "p", "n"), spins)[0]
    assert np.allclose(c, [1080, 1080, 0, 1080, 0])
    L, V = 2, 8
    rng = np.random.default_rng(9)
    s = {f: rng.standard_normal(V) + 1j * rng.standard_normal(V) for f in "uds"}
    S = {f: s[f][:, None, None] * np.eye(12)[None] for f in "uds"}
    F = _F(L, S, [("p", "n", "p", "n")])[0]
    a, b = s["u"] ** 2 * s["d"], s["u"] * s["d"] ** 2
    corr = np.array([np.sum(a[O._shift_index(L, r)] * b) for r in range(V)])
    ref = 1080 * np.einsum("ac,bd,r->abcdr", np.eye(4), np.eye(4), corr)
    assert _close(F, ref)


# ------------------------------------------------------------------ displacement orientation (L > 2)
# Reading A9 (eq. 2.1: B1 sits at X + r, B2 at X) and the q / -q pairing of eq. 2.6
# (PAPER.md:59).  At L = 2 every r equals -r and every twiddle is +-1, so the pins above cannot tell
# F(r) from F(-r); these run at L = 3 and 4, where r != -r, on channels with B1 != B2.
ASYM_CHANNELS = [("p", "L", "Sp", "n"), ("S0", "L", "Sp", "Sm"), ("Xm", "L", "S0", "Xm")]


def _site(L, x, y, z):
    return x + L * (y + L * z)


def test_orientation_tierA_equals_tierB_on_3cubed():
    """eq. 2.4 (direct X-sum, B1 at X + r) == eq. 2.6 (B~1(q) B~2(-q), inverse FFT) at every r of a 3^3
    lattice; F(r) != F(-r) there, so a swapped q <-> -q pairing or fft <-> ifft would fail."""
    L = 3
    S = rand_props(L, seed=31)
    bl = O.all_blocks(S, O.sink_names(ASYM_CHANNELS))
    FB = O.correlator_fft(L, bl, ASYM_CHANNELS)
    mr = O.minus_q_index(L)
    some = [_site(L, 1, 0, 0), _site(L, 2, 0, 0), _site(L, 1, 2, 0), _site(L, 2, 1, 0), _site(L, 0, 1, 2), _site(L, 0, 2, 1)]
    for ic, ch in enumerate(ASYM_CHANNELS):
        rs = list(range(L ** 3)) if ic == 0 else some  # every r for the first channel, three (r, -r) pairs for the others
        FA = O.correlator_direct(L, bl, ch, rs=rs)
        scale = abs(FA).max()
        assert abs(FA[..., rs] - FB[ic][..., rs]).max() <= 1e-13 * scale, ch
        # the test has teeth: the mirrored function is a different one
        assert abs(FB[ic][..., rs] - FB[ic][..., mr[rs]]).max() > 1e-2 * scale, ch


def test_orientation_two_site_support_4cubed():
    """Propagators supported on two sites x0, x1 of a 4^3 lattice: blocks live on those sites, so eq. 2.4 gives
    F(x0 - x1) = G(B1(x0), B2(x1)), F(x1 - x0) = G(B1(x1), B2(x0)), F(0) = G(x0, x0) + G(x1, x1) and zero at
    the other 61 displacements (G = pair_tensor, the site-local sum over P and xi').  r = x0 - x1 = (1, 3, 2)
    differs from -r = (3, 1, 2) (mod 4) on two axes.  Checked for tier A and tier B."""
    L, V = 4, 64
    x0, x1 = (2, 1, 3), (1, 2, 1)
    i0, i1 = _site(L, *x0), _site(L, *x1)
    r01 = _site(L, *[(a - b) % L for a, b in zip(x0, x1)])
    r10 = _site(L, *[(b - a) % L for a, b in zip(x0, x1)])
    assert r01 != r10 and r01 == _site(L, 1, 3, 2) and r10 == _site(L, 3, 1, 2)
    full = rand_props(L, seed=32)
    S = {f: np.zeros_like(full[f]) for f in "uds"}
    for f in "uds":
        S[f][[i0, i1]] = full[f][[i0, i1]]
    bl = O.all_blocks(S, O.sink_names(ASYM_CHANNELS))
    FB = O.correlator_fft(L, bl, ASYM_CHANNELS)
    for ic, ch in enumerate(ASYM_CHANNELS):
        B1, B2 = bl[ch[0]], bl[ch[1]]
        G = O.pair_tensor(B1[[i0, i1, i0, i1]], B2[[i1, i0, i0, i1]], ch)  # (x0,x1), (x1,x0), (x0,x0), (x1,x1)
        ref = np.zeros((4, 4, 4, 4, V), dtype=np.complex128)
        ref[..., r01] = G[0]
        ref[..., r10] = G[1]
        ref[..., 0] = G[2] + G[3]
        scale = abs(ref).max()
        assert abs(G[0] - G[1]).max() > 1e-2 * scale  # F(r01) and F(r10) are different numbers
        FA = O.correlator_direct(L, bl, ch, rs=[0, r01, r10, 1, 17, 63])
        for r in (0, r01, r10, 1, 17, 63):
            assert abs(FA[..., r] - ref[..., r]).max() <= 1e-13 * scale, (ch, r)
        assert abs(FB[ic] - ref).max() <= 1e-13 * scale, ch


def test_orientation_tierW_equals_tierA_on_3cubed():
    """Brute-force Wick contraction (oracle/wick.c: operators B1 at X + r, B2 at X, eq. 2.1) against tier A at
    asymmetric displacements of a 3^3 lattice, B1 != B2."""
    from oracle import wick
    L = 3
    S = rand_props(L, seed=33)
    ch = ("p", "L", "Sp", "n")
    spins = [(0, 1, 0, 1), (1, 0, 3, 2)]
    rs = [_site(L, 1, 0, 2), _site(L, 2, 0, 1), _site(L, 0, 1, 0)]  # r, -r, and another one
    bl = O.all_blocks(S, ch[:2])
    FA = O.correlator_direct(L, bl, ch, rs=rs)
    FW = wick.wick_fourpt(L, S, ch, spins, rs)
    FAs = np.array([[FA[s][r] for s in spins] for r in rs])
    scale = abs(FW).max()
    assert abs(FAs - FW).max() <= 1e-12 * scale
    assert abs(FW[0] - FW[1]).max() > 1e-2 * scale  # F(r) != F(-r)
