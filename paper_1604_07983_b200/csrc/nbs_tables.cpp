// Host table generator: channels -> sink pairs -> elementary correlators -> diagrams -> gather tables.
// Follows PAPER.md:45 (eq. 2.4), :57 (coset count), :67 (effective-block term count), :104-115
// (eqs. 4.2, 4.3) and the readings A1-A10 of DESIGN.md.  No code shared with oracle/.
#include "nbs_tables.hpp"

#include <algorithm>
#include <array>
#include <cmath>
#include <map>

namespace nbs {

namespace {

enum { U = 0, D = 1, S = 2 };

const double kS6 = 1.0 / std::sqrt(6.0);
const double kS2 = 1.0 / std::sqrt(2.0);

// eqs. 2.2-2.3 verbatim.  Block slot order: the operator's own field order for the octet members
// made of one elementary operator, (u, d, s) for Lambda, Sigma0 and the X's.
const BaryonDef kBaryons[NBS_NUM_BARYONS] = {
    /* p   */ {{U, D, U}, 1, {{+1.0, {U, D, U}}}},
    /* n   */ {{U, D, D}, 1, {{-1.0, {U, D, D}}}},
    /* L   */ {{U, D, S}, 3, {{kS6, {D, S, U}}, {kS6, {S, U, D}}, {-2.0 * kS6, {U, D, S}}}},
    /* S+  */ {{U, S, U}, 1, {{-1.0, {U, S, U}}}},
    /* S0  */ {{U, D, S}, 2, {{kS2, {D, S, U}}, {-kS2, {S, U, D}}}},
    /* S-  */ {{D, S, D}, 1, {{-1.0, {D, S, D}}}},
    /* X0  */ {{U, S, S}, 1, {{+1.0, {U, S, S}}}},
    /* X-  */ {{D, S, S}, 1, {{-1.0, {D, S, S}}}},
    /* Xu  */ {{U, D, S}, 1, {{+1.0, {D, S, U}}}},
    /* Xd  */ {{U, D, S}, 1, {{+1.0, {S, U, D}}}},
    /* Xs  */ {{U, D, S}, 1, {{+1.0, {U, D, S}}}},
};

int parity(const int* p, int n) {
    int inv = 0;
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j)
            if (p[i] > p[j]) ++inv;
    return (inv & 1) ? -1 : 1;
}

// Non-zeros of W[xi1 xi2 xi3; a] = eps_{c1c2c3} (C g5)_{a1a2} delta_{a3 a}  (reading A1 for C g5).
struct WEntry {
    int xi[3];
    int c[3];
    int a; // a3 = carried spin
    int sign;
};
std::vector<WEntry> w_nonzeros() {
    static const int cg5[4][3] = {{0, 1, +1}, {1, 0, -1}, {2, 3, +1}, {3, 2, -1}}; // (a1, a2, value)
    std::vector<WEntry> out;
    int c[3] = {0, 1, 2};
    do {
        int eps = parity(c, 3);
        for (auto& g : cg5)
            for (int a = 0; a < 4; ++a) {
                WEntry e;
                e.c[0] = c[0]; e.c[1] = c[1]; e.c[2] = c[2];
                e.xi[0] = c[0] + 3 * g[0];
                e.xi[1] = c[1] + 3 * g[1];
                e.xi[2] = c[2] + 3 * a;
                e.a = a;
                e.sign = eps * g[2];
                out.push_back(e);
            }
    } while (std::next_permutation(c, c + 3));
    return out;
}

// The factor of W that belongs to the sink baryon holding source positions `mask` (bit p-1 set
// <=> position p).  W = sum_shared factor(mask) * factor(7 ^ mask).
struct FactorEntry {
    int xi[3];  // value for each position held (-1 otherwise)
    int shared; // value of the shared index
    int carry;  // carried source spin (0 if this side does not hold position 3)
    int sign;
};
struct Factor {
    int nshared, ncarry;
    std::vector<FactorEntry> e;
};
Factor make_factor(int mask) {
    static const std::vector<WEntry> wnz = w_nonzeros();
    Factor f;
    f.ncarry = (mask & 4) ? 4 : 1;
    auto blank = [] { FactorEntry e; e.xi[0] = e.xi[1] = e.xi[2] = -1; e.shared = 0; e.carry = 0; e.sign = 1; return e; };
    switch (mask) {
    case 0:
        f.nshared = 1;
        f.e.push_back(blank());
        break;
    case 7: // whole source baryon on this side: full W, nothing shared
        f.nshared = 1;
        for (auto& w : wnz) {
            FactorEntry e = blank();
            e.xi[0] = w.xi[0]; e.xi[1] = w.xi[1]; e.xi[2] = w.xi[2];
            e.carry = w.a; e.sign = w.sign;
            f.e.push_back(e);
        }
        break;
    case 3: // the C g5 pair {1,2}: eps_{c1 c2 c} (C g5)_{a1 a2}, open colour c
        f.nshared = 3;
        for (auto& w : wnz) {
            if (w.a != 0) continue; // the delta on a3 belongs to the other side
            FactorEntry e = blank();
            e.xi[0] = w.xi[0]; e.xi[1] = w.xi[1];
            e.shared = w.c[2]; e.sign = w.sign;
            f.e.push_back(e);
        }
        break;
    case 4: // quark 3 alone: read at xi3 = (c, a), carries a
        f.nshared = 3;
        for (int c = 0; c < 3; ++c)
            for (int a = 0; a < 4; ++a) {
                FactorEntry e = blank();
                e.xi[2] = c + 3 * a; e.shared = c; e.carry = a;
                f.e.push_back(e);
            }
        break;
    case 5: // {1,3}: W with the partner index xi2 left open
    case 6: // {2,3}: W with the partner index xi1 left open
    {
        int open = (mask == 5) ? 1 : 0;
        f.nshared = NXI;
        for (auto& w : wnz) {
            FactorEntry e = blank();
            for (int p = 0; p < 3; ++p)
                if (p != open) e.xi[p] = w.xi[p];
            e.shared = w.xi[open]; e.carry = w.a; e.sign = w.sign;
            f.e.push_back(e);
        }
        break;
    }
    case 1: // lone C g5 partner: raw read at the shared index
    case 2: {
        int pos = (mask == 1) ? 0 : 1;
        f.nshared = NXI;
        for (int s = 0; s < NXI; ++s) {
            FactorEntry e = blank();
            e.xi[pos] = s; e.shared = s;
            f.e.push_back(e);
        }
        break;
    }
    }
    return f;
}
const Factor& factor(int mask) {
    static const std::array<Factor, 8> all = [] {
        std::array<Factor, 8> a;
        for (int m = 0; m < 8; ++m) a[m] = make_factor(m);
        return a;
    }();
    return all[mask];
}

// Gather table of one side of one diagram (eq. 4.2): slots[m] = source quark (0..5) in slot m.
struct SideTable {
    int C, K, n;
    int carries; // bit0: a3, bit1: a4
    std::vector<uint16_t> g;
};
SideTable make_side(const int* slots, int overall_sign, bool smem_layout = false) {
    int mask[2] = {0, 0};
    for (int m = 0; m < 3; ++m) mask[slots[m] / 3] |= 1 << (slots[m] % 3);
    const Factor& f0 = factor(mask[0]);
    const Factor& f1 = factor(mask[1]);
    SideTable t;
    t.C = f0.ncarry * f1.ncarry;
    t.K = f0.nshared * f1.nshared;
    t.carries = ((mask[0] & 4) ? 1 : 0) | ((mask[1] & 4) ? 2 : 0);
    size_t nent = (size_t)t.C * t.K;
    t.n = (int)(f0.e.size() * f1.e.size() / nent);
    std::vector<int> fill(nent, 0);
    t.g.assign(nent * t.n, 0);
    for (auto& e0 : f0.e)
        for (auto& e1 : f1.e) {
            int xi[3];
            for (int m = 0; m < 3; ++m) {
                int q = slots[m];
                xi[m] = (q / 3 == 0 ? e0 : e1).xi[q % 3];
            }
            int tri = smem_layout ? sm_index(xi[0], xi[1], xi[2]) : (xi[0] * NXI + xi[1]) * NXI + xi[2];
            int c = e0.carry * f1.ncarry + e1.carry;
            // shared index: the larger factor runs fastest (12 is a multiple of the MMA k-step 4, so
            // four consecutive k then differ in ONE colour-spin index: conflict-free gathers)
            int k = (f0.nshared > f1.nshared) ? e1.shared * f0.nshared + e0.shared
                                               : e0.shared * f1.nshared + e1.shared;
            int sign = e0.sign * e1.sign * overall_sign;
            size_t ent = (size_t)c * t.K + k;
            t.g[ent * t.n + fill[ent]++] = (uint16_t)(tri | (sign < 0 ? 0x8000 : 0));
        }
    return t;
}

struct RawDiagram {
    int P[6];
    int sign;
    double coef;
    int h[6]; // flavours of the six source quarks
};

std::string enumerate(const nbs_channel& ch, std::vector<RawDiagram>& out) {
    const int ids[4] = {ch.b1, ch.b2, ch.b3, ch.b4};
    for (int id : ids)
        if (id < 0 || id >= NBS_NUM_BARYONS) return "unknown baryon id";
    const BaryonDef &B1 = kBaryons[ch.b1], &B2 = kBaryons[ch.b2], &B3 = kBaryons[ch.b3], &B4 = kBaryons[ch.b4];
    int g[6];
    for (int j = 0; j < 3; ++j) { g[j] = B1.slot[j]; g[3 + j] = B2.slot[j]; }
    for (int i3 = 0; i3 < B3.nterm; ++i3)
        for (int i4 = 0; i4 < B4.nterm; ++i4) {
            RawDiagram d;
            for (int j = 0; j < 3; ++j) { d.h[j] = B3.term[i3].f[j]; d.h[3 + j] = B4.term[i4].f[j]; }
            d.coef = B3.term[i3].coef * B4.term[i4].coef;
            int P[6] = {0, 1, 2, 3, 4, 5};
            do {
                bool ok = true;
                for (int j = 0; j < 6 && ok; ++j) ok = (g[j] == d.h[P[j]]);
                // one representative per coset modulo exchange of same-flavour slots inside one
                // sink baryon (the block is antisymmetric there): the paper's 2^{N_L+N_S0-B}
                for (int base = 0; base < 6 && ok; base += 3)
                    for (int j = base; j < base + 3 && ok; ++j)
                        for (int k = j + 1; k < base + 3 && ok; ++k)
                            if (g[j] == g[k] && P[j] > P[k]) ok = false;
                if (!ok) continue;
                for (int j = 0; j < 6; ++j) d.P[j] = P[j];
                d.sign = parity(P, 6);
                out.push_back(d);
            } while (std::next_permutation(P, P + 6));
        }
    if (out.empty()) return "channel violates flavour conservation (F vanishes identically)";
    return "";
}

int diagram_K(const int* P) {
    int mask[2] = {0, 0};
    for (int m = 0; m < 3; ++m) mask[P[m] / 3] |= 1 << (P[m] % 3);
    return factor(mask[0]).nshared * factor(mask[1]).nshared;
}

} // namespace

const BaryonDef& baryon_def(int id) { return kBaryons[id]; }

int baryon_iso_mirror(int baryon, int* eta) {
    const BaryonDef& B = kBaryons[baryon];
    auto flip = [](int f) { return f == U ? D : f == D ? U : f; };
    for (int cand = 0; cand < NBS_NUM_BARYONS; ++cand) {
        const BaryonDef& Bc = kBaryons[cand];
        if (Bc.nterm != B.nterm) continue;
        for (int e = +1; e >= -1; e -= 2) {
            bool all = true;
            for (int i = 0; i < B.nterm && all; ++i) {
                // image of term i: coef * eps (q_f0' C g5 q_f1') q_f2'  =  -coef * eps (q_f1' C g5 q_f0') q_f2'
                const int f0 = flip(B.term[i].f[0]), f1 = flip(B.term[i].f[1]), f2 = flip(B.term[i].f[2]);
                bool found = false;
                for (int j = 0; j < Bc.nterm && !found; ++j) {
                    const ElemTerm& t = Bc.term[j];
                    if (t.f[2] != f2) continue;
                    if (t.f[0] == f0 && t.f[1] == f1 && std::fabs(e * t.coef - B.term[i].coef) < 1e-14) found = true;
                    if (t.f[0] == f1 && t.f[1] == f0 && std::fabs(e * t.coef + B.term[i].coef) < 1e-14) found = true;
                }
                all = found;
            }
            if (all) { if (eta) *eta = e; return cand; }
        }
    }
    return -1;
}

std::vector<IsoRelation> iso_channel_relations(const std::vector<nbs_channel>& channels) {
    std::vector<IsoRelation> rel(channels.size(), IsoRelation{-1, 1, 0});
    std::vector<char> has_alias(channels.size(), 0);
    for (size_t i = 0; i < channels.size(); ++i) {
        if (rel[i].from >= 0 || has_alias[i]) continue;
        const nbs_channel& c = channels[i];
        int e1, e2, e3, e4;
        const int m1 = baryon_iso_mirror(c.b1, &e1), m2 = baryon_iso_mirror(c.b2, &e2), m3 = baryon_iso_mirror(c.b3, &e3),
                  m4 = baryon_iso_mirror(c.b4, &e4);
        if (m1 < 0 || m2 < 0 || m3 < 0 || m4 < 0) continue;
        const int s = e1 * e2 * e3 * e4;
        for (size_t j = i + 1; j < channels.size(); ++j) {
            if (rel[j].from >= 0 || has_alias[j]) continue;
            const nbs_channel& d = channels[j];
            if (d.b1 != m1 || d.b2 != m2) continue;
            if (d.b3 == m3 && d.b4 == m4) { rel[j] = IsoRelation{(int)i, s, 0}; has_alias[i] = 1; break; }
            if (d.b3 == m4 && d.b4 == m3) { rel[j] = IsoRelation{(int)i, -s, 1}; has_alias[i] = 1; break; }
        }
    }
    return rel;
}

int block_kind(int baryon) {
    const BaryonDef& B = kBaryons[baryon];
    if (B.slot[0] == B.slot[2]) return BK_ASYM13;
    if (B.slot[1] == B.slot[2]) return BK_ASYM23;
    return BK_FULL;
}

std::vector<BlockTerm> block_terms(int baryon) {
    const BaryonDef& B = kBaryons[baryon];
    std::vector<BlockTerm> out;
    for (int i = 0; i < B.nterm; ++i) {
        int sig[3] = {0, 1, 2};
        do { // Wick pairings: field j -> slot sig[j] of the same flavour, sign sgn(sig)
            bool ok = true;
            for (int j = 0; j < 3; ++j) ok = ok && (B.term[i].f[j] == B.slot[sig[j]]);
            if (!ok) continue;
            BlockTerm t;
            t.coef = B.term[i].coef * parity(sig, 3);
            t.f0 = B.term[i].f[0]; t.f1 = B.term[i].f[1]; t.f2 = B.term[i].f[2];
            for (int j = 0; j < 3; ++j) t.perm[j] = sig[j];
            out.push_back(t);
        } while (std::next_permutation(sig, sig + 3));
    }
    return out;
}

std::vector<nbs_channel> standard_channels() {
    // Reading A10: sectors of fixed strangeness and charge, all sink x source pairs inside a
    // sector except the four isospin-forbidden LL <-> S0L and S0S0 <-> S0L.
    typedef std::pair<int, int> St;
    const std::vector<std::vector<St>> sectors = {
        {{NBS_P, NBS_N}},
        {{NBS_P, NBS_LAMBDA}, {NBS_SIGMA_P, NBS_N}, {NBS_SIGMA_0, NBS_P}},
        {{NBS_LAMBDA, NBS_LAMBDA}, {NBS_P, NBS_XI_M}, {NBS_N, NBS_XI_0}, {NBS_SIGMA_P, NBS_SIGMA_M},
         {NBS_SIGMA_0, NBS_SIGMA_0}, {NBS_SIGMA_0, NBS_LAMBDA}},
        {{NBS_XI_M, NBS_LAMBDA}, {NBS_SIGMA_M, NBS_XI_0}, {NBS_SIGMA_0, NBS_XI_M}},
        {{NBS_XI_M, NBS_XI_0}},
    };
    const St LL{NBS_LAMBDA, NBS_LAMBDA}, S0L{NBS_SIGMA_0, NBS_LAMBDA}, S0S0{NBS_SIGMA_0, NBS_SIGMA_0};
    std::vector<nbs_channel> out;
    for (auto& sec : sectors)
        for (auto& snk : sec)
            for (auto& src : sec) {
                bool forbidden = (snk == S0L && (src == LL || src == S0S0)) || (src == S0L && (snk == LL || snk == S0S0));
                if (forbidden) continue;
                out.push_back(nbs_channel{snk.first, snk.second, src.first, src.second});
            }
    return out;
}

std::string channel_diagrams(const nbs_channel& ch, std::vector<DiagramInfo>& out) {
    std::vector<RawDiagram> raw;
    std::string err = enumerate(ch, raw);
    if (!err.empty()) return err;
    for (auto& d : raw) {
        DiagramInfo di;
        for (int j = 0; j < 6; ++j) di.P[j] = d.P[j];
        di.sign = d.sign;
        di.K = diagram_K(d.P);
        out.push_back(di);
    }
    return "";
}

std::string build_plan(const std::vector<nbs_channel>& channels, Plan& plan, int unit_split_steps, int unit_cost_max,
                       const std::vector<char>* iso_conj) {
    plan = Plan();
    plan.channels = channels;
    if (channels.empty()) return "empty channel list";

    // sink pairs in order of first appearance; needed baryon blocks
    std::map<std::pair<int, int>, int> pair_index;
    std::vector<std::pair<int, int>> pair_list;
    std::map<int, int> slot_of;
    auto slot = [&](int b) {
        auto it = slot_of.find(b);
        if (it != slot_of.end()) return it->second;
        int s = (int)plan.baryons.size();
        plan.baryons.push_back(b);
        slot_of[b] = s;
        return s;
    };
    // elementary correlators per pair, keyed by the six source flavours
    typedef std::array<int, 6> Key;
    std::vector<std::map<Key, std::vector<RawDiagram>>> pair_elems;
    std::vector<std::vector<Key>> pair_elem_order;
    struct CT { int pair; Key key; double coef; };
    std::vector<std::vector<CT>> chan_ct(channels.size());

    for (size_t ic = 0; ic < channels.size(); ++ic) {
        const nbs_channel& ch = channels[ic];
        std::vector<RawDiagram> raw;
        std::string err = enumerate(ch, raw);
        if (!err.empty()) return "channel " + std::to_string(ic) + ": " + err;
        auto pk = std::make_pair(ch.b1, ch.b2);
        int ip;
        if (!pair_index.count(pk)) {
            ip = (int)pair_list.size();
            pair_index[pk] = ip;
            pair_list.push_back(pk);
            pair_elems.emplace_back();
            pair_elem_order.emplace_back();
            slot(ch.b1); slot(ch.b2);
        } else ip = pair_index[pk];
        plan.chan_pair.push_back(ip);
        std::map<Key, std::vector<RawDiagram>> mine;
        std::vector<Key> order;
        for (auto& d : raw) {
            Key k; for (int j = 0; j < 6; ++j) k[j] = d.h[j];
            if (!mine.count(k)) order.push_back(k);
            mine[k].push_back(d);
            plan.sumK_std += diagram_K(d.P);
        }
        for (auto& k : order) {
            if (!pair_elems[ip].count(k)) {
                pair_elems[ip][k] = mine[k];
                pair_elem_order[ip].push_back(k);
            }
            chan_ct[ic].push_back(CT{ip, k, mine[k][0].coef});
        }
    }

    // Source-swap reduction (reading A11): exchanging the two source operators gives
    //   E[B3 B4]_{a1 a2 a3 a4} = - E[B4 B3]_{a1 a2 a4 a3},
    // so of two elementary correlators of one sink pair whose source operators are each other's
    // swap only the lexicographically smaller key is computed; the epilogue reads the other one
    // from it with a3 <-> a4 exchanged and the sign flipped.
    auto swapped = [](const Key& k) { return Key{k[3], k[4], k[5], k[0], k[1], k[2]}; };
    std::vector<std::vector<Key>> pair_comp_order(pair_list.size()); // computed keys
    for (size_t ip = 0; ip < pair_list.size(); ++ip)
        for (auto& k : pair_elem_order[ip]) {
            const Key ks = swapped(k);
            const bool derived = ks != k && pair_elems[ip].count(ks) && ks < k;
            if (!derived) pair_comp_order[ip].push_back(k);
        }

    // slot order: baryons whose block follows from a partner's in the isospin limit (n from p, Sigma- from
    // Sigma+, Xi- from Xi0) go last, so that the fast path works on a prefix of the row
    auto iso_partner = [&](int b) {
        const int partner = (b == NBS_N) ? NBS_P : (b == NBS_SIGMA_M) ? NBS_SIGMA_P : (b == NBS_XI_M) ? NBS_XI_0 : -1;
        return (partner >= 0 && slot_of.count(partner)) ? partner : -1;
    };
    {
        std::vector<int> ordered;
        for (int b : plan.baryons) if (iso_partner(b) < 0) ordered.push_back(b);
        plan.n_slots_iso = (int)ordered.size();
        for (int b : plan.baryons) if (iso_partner(b) >= 0) ordered.push_back(b);
        plan.baryons = ordered;
        for (size_t i = 0; i < ordered.size(); ++i) slot_of[ordered[i]] = (int)i;
    }

    // compact site row; expansion map of the antisymmetric slots into full staged blocks
    for (size_t sl = 0; sl < plan.baryons.size(); ++sl) {
        const int kind = block_kind(plan.baryons[sl]);
        const int base = plan.row_elems;
        plan.slot_off.push_back(base);
        plan.slot_kind.push_back(kind);
        plan.row_elems += block_elems(kind);
        if (kind == BK_FULL) { plan.slot_src.push_back(int2x{0, base}); continue; }
        const int ebase = plan.n_asym * SM_BLOCK;
        plan.slot_src.push_back(int2x{1, ebase});
        ++plan.n_asym;
        plan.gather.resize(ebase + SM_BLOCK, -1);
        for (int al = 0; al < 4; ++al)
            for (int x1 = 0; x1 < NXI; ++x1)
                for (int x2 = 0; x2 < NXI; ++x2)
                    for (int x3 = 0; x3 < NXI; ++x3) {
                        if ((kind == BK_ASYM13 ? x1 : x2) == x3) continue; // diagonal: zero
                        const Located loc = locate(kind, x1, x2, x3);
                        const int src = base + al * AS_PLANE + loc.idx;
                        plan.gather[ebase + al * SM_PLANE + sm_index(x1, x2, x3)] = src | (loc.sign < 0 ? (1 << 30) : 0);
                    }
    }

    // expansion map of the isospin-limit fast path: derived slots gather from their partner's compact block
    plan.gather_iso = plan.gather;
    plan.row_elems_iso = plan.n_slots_iso < (int)plan.baryons.size() ? plan.slot_off[plan.n_slots_iso] : plan.row_elems;
    for (size_t sl = plan.n_slots_iso; sl < plan.baryons.size(); ++sl) {
        const int b = plan.baryons[sl], partner = iso_partner(b);
        const int pbase = plan.slot_off[slot_of[partner]], pkind = block_kind(partner);
        const int ebase = plan.slot_src[sl].y;
        for (int al = 0; al < 4; ++al)
            for (int x1 = 0; x1 < NXI; ++x1)
                for (int x2 = 0; x2 < NXI; ++x2)
                    for (int x3 = 0; x3 < NXI; ++x3) {
                        // n(x1 x2 x3) = -p(x2 x1 x3);  Sigma-(x) = Sigma+(x);  Xi-(x) = -Xi0(x)
                        const bool tr = (b == NBS_N);
                        const int y1 = tr ? x2 : x1, y2 = tr ? x1 : x2;
                        const int sign = (b == NBS_SIGMA_M) ? +1 : -1;
                        int& g = plan.gather_iso[ebase + al * SM_PLANE + sm_index(x1, x2, x3)];
                        if ((pkind == BK_ASYM13 ? y1 : y2) == x3) { g = -1; continue; } // partner's diagonal: zero
                        const Located loc = locate(pkind, y1, y2, x3);
                        g = (pbase + al * AS_PLANE + loc.idx) | ((sign * loc.sign < 0) ? (1 << 30) : 0);
                    }
    }

    // ---- product kernel tables: pairs -> (<= MAX_PAIR_ELEMS elementary correlators) -> units -> diagrams
    // layout: 0 = 16x16 side, 1 = 64x4 A side, 2 = 64x4 B side (see nbs_tables.hpp)
    std::map<std::vector<uint32_t>, uint32_t> dedupe3;
    std::string tab_err;
    auto intern3 = [&](const SideTable& t, int layout) -> uint32_t {
        const int Kp = (t.K + 3) / 4 * 4, nw = t.n / 2;
        const int rows = (layout == 2) ? 4 : 8, G = (layout == 1) ? 4 : 1;
        // padded k (k >= K): off+ == off- == 0.  One extra all-zero k-step closes every table: the
        // kernel's software pipeline gathers one k-step past the end of a unit's range, and those
        // (unused) gathers must not pick up offsets of a following table with another layout.
        std::vector<uint32_t> w((size_t)(Kp + 4) * rows * G * nw * 2, 0u);
        for (int k = 0; k < t.K; ++k)
            for (int r = 0; r < rows; ++r)
                for (int g = 0; g < G; ++g) {
                    // carried index and sink-spin plane folded into the byte offset
                    const int c = (layout == 0) ? (r >> 1) : (layout == 1) ? 4 * g + (r >> 1) : 0;
                    const int plane = (layout == 2) ? r : (r & 1);
                    std::vector<uint32_t> plus, minus;
                    for (int j = 0; j < t.n; ++j) {
                        const uint16_t e = t.g[((size_t)c * t.K + k) * t.n + j];
                        const uint32_t off = (uint32_t)(plane * SM_PLANE + (e & 0x7fff)) * 16u;
                        ((e & 0x8000) ? minus : plus).push_back(off);
                    }
                    if ((int)plus.size() != nw || (int)minus.size() != nw) { tab_err = "internal: unbalanced gather signs"; return 0; }
                    for (int j = 0; j < nw; ++j) {
                        const size_t o = ((((size_t)k * rows + r) * G + g) * nw + j) * 2;
                        w[o] = plus[j]; w[o + 1] = minus[j];
                    }
                }
        w.push_back((uint32_t)layout); // same content in another layout is another table
        auto it = dedupe3.find(w);
        if (it != dedupe3.end()) return it->second;
        w.pop_back();
        const uint32_t off = (uint32_t)plan.tab3.size();
        for (size_t i = 0; i < w.size(); i += 2) plan.tab3.push_back(uint2x{w[i], w[i + 1]});
        while (plan.tab3.size() % 2) plan.tab3.push_back(uint2x{0, 0}); // 16-byte aligned tables
        w.push_back((uint32_t)layout);
        dedupe3[w] = off;
        return off;
    };
    // Tables of the pipelined kernel (nbs_tables.hpp, "packed gather tables"): one 32-bit word per term pair,
    // offsets inside ONE sink-spin plane of a block of kind `kind` (raw index triples from make_side).  An
    // antisymmetric block is gathered from its compact form: a term whose stored partner carries the opposite sign
    // changes sides (u <-> v); when an entry then has more terms of one sign than it has places for, the surplus
    // goes to the other side with its flip bit set; the vanishing diagonal is read from a zero pad.
    std::map<std::vector<uint32_t>, uint32_t> dedupec;
    auto intern3c = [&](const SideTable& t, int layout, int kind) -> uint32_t {
        const int Kp = (t.K + 3) / 4 * 4, nw = t.n / 2;
        const int G = (layout == 1) ? 4 : 1, CC = (layout == 2) ? 1 : 4;
        // C_TAB_LOOKAHEAD all-zero k-steps close every table: the kernel's software pipeline reads that far past
        // the end of a unit's range, and a zero word gathers u = v = entry 0 of the plane (difference 0)
        std::vector<uint32_t> w((size_t)(Kp + 4 * C_TAB_LOOKAHEAD) * CC * G * nw, 0u);
        for (int k = 0; k < t.K; ++k)
            for (int cc = 0; cc < CC; ++cc)
                for (int g = 0; g < G; ++g) {
                    const int c = (layout == 0) ? cc : (layout == 1) ? 4 * g + cc : 0; // carried source spin(s)
                    std::vector<uint32_t> plus, minus, zeros;
                    for (int j = 0; j < t.n; ++j) {
                        const uint16_t e = t.g[((size_t)c * t.K + k) * t.n + j];
                        const int tri = e & 0x7fff, sg = (e & 0x8000) ? -1 : 1;
                        const Located loc = locate(kind, tri / 144, (tri / 12) % 12, tri % 12);
                        const uint32_t off = (uint32_t)loc.idx * 16u; // < 2^15
                        if (loc.sign == 0) zeros.push_back(off);
                        else ((sg * loc.sign < 0) ? minus : plus).push_back(off);
                    }
                    std::vector<uint32_t> U, V; // 16-bit halves: byte offset | flip << 15
                    for (uint32_t o : plus) { if ((int)U.size() < nw) U.push_back(o); else V.push_back(o | 0x8000u); }
                    for (uint32_t o : minus) { if ((int)V.size() < nw) V.push_back(o); else U.push_back(o | 0x8000u); }
                    for (uint32_t o : zeros) { if ((int)U.size() < nw) U.push_back(o); else V.push_back(o); }
                    if ((int)U.size() != nw || (int)V.size() != nw) { tab_err = "internal: compact gather does not fit"; return 0; }
                    for (int j = 0; j < nw; ++j) {
                        // layout 0: [k][c][nw]; layout 1: [k][cX & 3][g]; layout 2: [k][nw]
                        const size_t o = (layout == 1) ? ((size_t)k * 4 + cc) * 4 + g : ((size_t)k * CC + cc) * nw + j;
                        w[o] = U[j] | (V[j] << 16);
                    }
                }
        w.push_back((uint32_t)layout);
        auto it = dedupec.find(w);
        if (it != dedupec.end()) return it->second;
        w.pop_back();
        const uint32_t off = (uint32_t)plan.tabc.size();
        plan.tabc.insert(plan.tabc.end(), w.begin(), w.end());
        while (plan.tabc.size() % 4) plan.tabc.push_back(0u); // 16-byte aligned tables
        w.push_back((uint32_t)layout);
        dedupec[w] = off;
        return off;
    };
    const int UNIT_SPLIT_STEPS = unit_split_steps, UNIT_COST_MAX = unit_cost_max; // cost: 2 per 16x16 step, 3 per 64x4 step
    for (size_t ip = 0; ip < pair_list.size(); ++ip) {
        const std::vector<Key>& order = pair_comp_order[ip];
        // at most 15 distinct elementary source operator pairs share the flavour content of one sink pair
        if (order.size() > (size_t)MAX_PAIR_ELEMS) return "internal: more than 16 elementary correlators for one sink pair";
        Pair3Rec pr;
        pr.slot1 = slot_of[pair_list[ip].first];
        pr.slot2 = slot_of[pair_list[ip].second];
        pr.unit_begin = (int)plan.units3.size();
        pr.diag_begin = (int)plan.diags3.size();
        pr.nelem = (int)order.size();
        pr.swap_mask = 0;
        pr.self_swap = (pair_list[ip].first == pair_list[ip].second) ? 1 : 0;
        std::vector<Unit3Rec> units;
        std::vector<int> cost_of;
        for (size_t e = 0; e < order.size(); ++e) {
            pr.elem_unit_begin[e] = (int)units.size();
            for (int cls = 0; cls < 4; ++cls) {
                Unit3Rec u;
                int ucost = 0;
                u.cls = cls; u.diag_begin = (int)plan.diags3.size() - pr.diag_begin;
                auto flush = [&] {
                    u.diag_end = (int)plan.diags3.size() - pr.diag_begin;
                    if (u.diag_end > u.diag_begin) { u.slot = (int)units.size(); units.push_back(u); cost_of.push_back(ucost); }
                    u.diag_begin = u.diag_end; ucost = 0;
                };
                for (auto& d : pair_elems[ip][order[e]]) {
                    SideTable s1 = make_side(d.P, d.sign, true); // sigma_P folded into side 1
                    SideTable s2 = make_side(d.P + 3, +1, true);
                    int c;
                    if (s1.C == 4 && s2.C == 4) c = (s1.carries == 1) ? 0 : 1;
                    else if (s1.C == 16 && s2.C == 1) c = 2;
                    else if (s1.C == 1 && s2.C == 16) c = 3;
                    else return "internal: unexpected carry split";
                    if (c != cls) continue;
                    if ((s1.n & 1) || (s2.n & 1)) return "internal: odd gather length";
                    const SideTable &A = (c == 3) ? s2 : s1, &B = (c == 3) ? s1 : s2;
                    if (c < 2 ? !(A.n == B.n && (A.n == 2 || A.n == 8 || A.n == 24)) : !(A.n == 2 && B.n == 8))
                        return "internal: unexpected gather lengths";
                    Diag3Rec r, rc;
                    r.offA = intern3(A, c < 2 ? 0 : 1); r.offB = intern3(B, c < 2 ? 0 : 2);
                    {
                        const SideTable r1 = make_side(d.P, d.sign, false), r2 = make_side(d.P + 3, +1, false);
                        const int k1 = block_kind(pair_list[ip].first), k2 = block_kind(pair_list[ip].second);
                        const SideTable &Ar = (c == 3) ? r2 : r1, &Br = (c == 3) ? r1 : r2;
                        rc.offA = intern3c(Ar, c < 2 ? 0 : 1, (c == 3) ? k2 : k1);
                        rc.offB = intern3c(Br, c < 2 ? 0 : 2, (c == 3) ? k1 : k2);
                    }
                    if (!tab_err.empty()) return tab_err;
                    r.K = (uint16_t)s1.K;
                    (pr.self_swap ? plan.sumK_exec_self : plan.sumK_exec) += s1.K;
                    r.nwA = (uint8_t)(A.n / 2); r.nwB = (uint8_t)(B.n / 2);
                    // split long diagrams into k-ranges so that a sink pair with few diagrams
                    // still spreads over all warps of the CTA
                    const int steps = (s1.K + 3) / 4;
                    const int nchunk = (steps + UNIT_SPLIT_STEPS - 1) / UNIT_SPLIT_STEPS;
                    for (int ic = 0; ic < nchunk; ++ic) {
                        const int sb = steps * ic / nchunk, se = steps * (ic + 1) / nchunk;
                        r.sbeg = (uint16_t)sb; r.send = (uint16_t)se;
                        const int cost = (se - sb) * (c >= 2 ? 3 : 2) * (c < 2 ? (int)r.nwA : 1) + 2;
                        if (ucost > 0 && ucost + cost > UNIT_COST_MAX) flush();
                        plan.diags3.push_back(r);
                        rc.K = r.K; rc.nwA = r.nwA; rc.nwB = r.nwB; rc.sbeg = r.sbeg; rc.send = r.send;
                        plan.diagsc.push_back(rc);
                        ucost += cost;
                        plan.sumKp_exec += 4 * (se - sb);
                    }
                }
                flush();
            }
        }
        pr.nunits = (int)units.size();
        pr.ndiags = (int)plan.diags3.size() - pr.diag_begin;
        if (pr.nunits > MAX_PAIR_UNITS || pr.ndiags > MAX_PAIR_DIAGS) return "internal: too many units for one sink pair";
        for (int e = pr.nelem; e <= MAX_PAIR_ELEMS; ++e) pr.elem_unit_begin[e] = pr.nunits;
        plan.max_pair_units = std::max(plan.max_pair_units, pr.nunits);
        plan.max_pair_diags = std::max(plan.max_pair_diags, pr.ndiags);
        // schedule: units by decreasing cost (warps take them in this order)
        std::vector<int> idx(pr.nunits);
        for (int i = 0; i < pr.nunits; ++i) idx[i] = i;
        std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return cost_of[a] > cost_of[b]; });
        for (int i : idx) plan.units3.push_back(units[i]);
        // channels of this pair as dense coefficient rows over its elementary correlators
        pr.chan_begin = (int)plan.pair_chans.size();
        for (size_t ic = 0; ic < channels.size(); ++ic) {
            if (plan.chan_pair[ic] != (int)ip) continue;
            PairChanRec pc;
            pc.ch = (int)ic; pc.local = (int)plan.pair_chans.size() - pr.chan_begin;
            pc.alias_ch = -1; pc.alias_swap = 0; pc.alias_sign = 1.0;
            pc.mirror_ch = pc.ch; pc.mirror_swap = 0; pc.mirror_sign = -1.0;
            bool any = false;
            for (int e = 0; e < MAX_PAIR_ELEMS; ++e) pc.coef[e] = pc.coefS[e] = 0.0;
            for (auto& ct : chan_ct[ic])
                for (size_t e = 0; e < order.size(); ++e) {
                    if (order[e] == ct.key) { pc.coef[e] += ct.coef; any = true; }
                    else if (order[e] == swapped(ct.key)) { // derived: - (computed one with a3 <-> a4)
                        pc.coefS[e] -= ct.coef; any = true;
                        pr.swap_mask |= 1 << e;
                    }
                }
            if (any) plan.pair_chans.push_back(pc);
        }
        pr.nchan = (int)plan.pair_chans.size() - pr.chan_begin;
        // isospin limit: sink pair of a field and its u <-> d image, channel set closed under the images of the sources
        if (iso_conj && !pr.self_swap) {
            const int b1 = pair_list[ip].first, b2 = pair_list[ip].second;
            int e1 = 0, e2 = 0;
            bool ok = baryon_iso_mirror(b1, &e1) == b2 && baryon_iso_mirror(b2, &e2) == b1 && pr.nchan > 0;
            std::vector<PairChanRec> recs(plan.pair_chans.begin() + pr.chan_begin, plan.pair_chans.end());
            // the relation pairs the channel records up (a record may be its own partner); a list may hold a channel twice
            std::vector<char> matched(recs.size(), 0);
            for (size_t i = 0; i < recs.size() && ok; ++i) {
                if (matched[i]) continue;
                PairChanRec& pc = recs[i];
                const nbs_channel& c = channels[pc.ch];
                int e3 = 0, e4 = 0;
                const int m3 = baryon_iso_mirror(c.b3, &e3), m4 = baryon_iso_mirror(c.b4, &e4);
                ok = m3 >= 0 && m4 >= 0 && !(*iso_conj)[pc.ch];
                if (!ok) break;
                const int s = e1 * e2 * e3 * e4;
                auto relation = [&](const nbs_channel& d, int& swap, double& sign) {
                    if (d.b3 == m3 && d.b4 == m4) { swap = 0; sign = -(double)s; return true; }
                    if (d.b3 == m4 && d.b4 == m3) { swap = 1; sign = (double)s; return true; }
                    return false;
                };
                int swap = 0;
                double sign = 0.0;
                size_t j = recs.size();
                if (relation(c, swap, sign)) j = i; // its own partner
                else
                    for (size_t k = i + 1; k < recs.size(); ++k)
                        if (!matched[k] && !(*iso_conj)[recs[k].ch] && relation(channels[recs[k].ch], swap, sign)) { j = k; break; }
                ok = j < recs.size();
                if (!ok) break;
                pc.mirror_ch = recs[j].ch; pc.mirror_swap = swap; pc.mirror_sign = sign;
                recs[j].mirror_ch = pc.ch; recs[j].mirror_swap = swap; recs[j].mirror_sign = sign;
                matched[i] = matched[j] = 1;
            }
            if (ok) {
                std::copy(recs.begin(), recs.end(), plan.pair_chans.begin() + pr.chan_begin);
                pr.self_swap = 2;
            }
        }
        plan.pairs3.push_back(pr);
    }
    plan.tab3.insert(plan.tab3.end(), 4096, uint2x{0, 0}); // the kernel prefetches a few k-steps past a table's end (4096: also covers nbs_plan_selfcheck's class-blind bound)
    plan.tabc.insert(plan.tabc.end(), 256, 0u); // L1 prefetches run a little past a table's end

    // ---- chains: order of the sink pairs inside one momentum task that reloads the fewest blocks.
    // Full chain (all pairs) for the momenta q <= -q (index order), half chain (without the pairs of
    // identical sink baryons) for the others: for B1 == B2 the sink-swap relation (DESIGN.md reading
    // A11)  F~_{a1 a2 ..}(-q) = - F~_{a2 a1 ..}(q)  gives the -q result from the q result.
    auto make_chain = [&](const std::vector<int>& ids) {
        const int n = (int)ids.size();
        // cost of walking from pair a to pair b: block slots to stage, plus a penalty when the new
        // blocks do not fit beside those of a in the four shared-memory slots of the pipelined kernel -- such a
        // transition cannot be prefetched: the loads wait for a to complete and every warp waits for the loads
        auto nsl = [&](int slot) { return plan.slot_kind[slot] == BK_FULL ? 2 : 1; };
        auto tcost = [&](int a, int b) {
            const Pair3Rec &pa = plan.pairs3[ids[a]], &pb = plan.pairs3[ids[b]];
            const int used = nsl(pa.slot1) + nsl(pa.slot2);
            const int fresh = (pa.slot1 != pb.slot1 ? nsl(pb.slot1) : 0) + (pa.slot2 != pb.slot2 ? nsl(pb.slot2) : 0);
            return fresh + (fresh > C_NSLOT - used ? 8 : 0);
        };
        std::vector<int> best;
        if (n == 0) return;
        if (n <= 16) { // exact: shortest Hamiltonian path by subset DP
            const int N = 1 << n, INF = 1 << 28;
            std::vector<int> dp((size_t)N * n, INF), from((size_t)N * n, -1);
            for (int i = 0; i < n; ++i) dp[((size_t)1 << i) * n + i] = nsl(plan.pairs3[ids[i]].slot1) + nsl(plan.pairs3[ids[i]].slot2);
            for (int m = 1; m < N; ++m)
                for (int i = 0; i < n; ++i) {
                    const int cur = dp[(size_t)m * n + i];
                    if (cur >= INF || !((m >> i) & 1)) continue;
                    for (int j = 0; j < n; ++j) {
                        if ((m >> j) & 1) continue;
                        const int m2 = m | (1 << j), c = cur + tcost(i, j);
                        if (c < dp[(size_t)m2 * n + j]) { dp[(size_t)m2 * n + j] = c; from[(size_t)m2 * n + j] = i; }
                    }
                }
            int bi = 0;
            for (int i = 1; i < n; ++i)
                if (dp[(size_t)(N - 1) * n + i] < dp[(size_t)(N - 1) * n + bi]) bi = i;
            int m = N - 1, i = bi;
            while (i >= 0) { best.push_back(i); const int pi = from[(size_t)m * n + i]; m &= ~(1 << i); i = pi; }
            std::reverse(best.begin(), best.end());
        } else { // greedy nearest neighbour
            std::vector<char> used(n, 0);
            int cur = 0;
            used[0] = 1; best.push_back(0);
            for (int s = 1; s < n; ++s) {
                int bj = -1;
                for (int j = 0; j < n; ++j)
                    if (!used[j] && (bj < 0 || tcost(cur, j) < tcost(cur, bj))) bj = j;
                used[bj] = 1; best.push_back(bj); cur = bj;
            }
        }
        for (int s = 0; s < n; ++s) {
            ChainRec cr;
            cr.pair = ids[best[s]];
            cr.load1 = (s == 0) || plan.pairs3[cr.pair].slot1 != plan.pairs3[ids[best[s - 1]]].slot1;
            cr.load2 = (s == 0) || plan.pairs3[cr.pair].slot2 != plan.pairs3[ids[best[s - 1]]].slot2;
            const Pair3Rec& pr = plan.pairs3[cr.pair];
            cr.nunits = pr.nunits; cr.unit_begin = pr.unit_begin; cr.ndiags = pr.ndiags; cr.diag_begin = pr.diag_begin; cr.pad = 0;
            cr.buf1 = plan.slot_src[pr.slot1].x; cr.off1 = plan.slot_src[pr.slot1].y;
            cr.buf2 = plan.slot_src[pr.slot2].x; cr.off2 = plan.slot_src[pr.slot2].y;
            plan.chain.push_back(cr);
        }
    };
    {
        std::vector<int> all, half;
        for (int i = 0; i < (int)plan.pairs3.size(); ++i) {
            all.push_back(i);
            if (!plan.pairs3[i].self_swap) half.push_back(i);
        }
        make_chain(all);
        plan.chain_full_n = (int)plan.chain.size();
        make_chain(half);
        plan.chain_half_n = (int)plan.chain.size() - plan.chain_full_n;
        plan.chain_single_begin = (int)plan.chain.size();
        for (int i = 0; i < (int)plan.pairs3.size(); ++i) make_chain(std::vector<int>{i});
    }
    // isospin limit: the compact blocks of the derived slots are those of their partners up to a sign
    //   n(x1 x2 x3) = -p(x2 x1 x3): the compact entry [xi_c = x1][pair (x2, x3)] of n is minus the compact entry
    //   [xi_c = x1][pair (x2', x3)] of p with its antisymmetric pair (x1', x3) = (x2, x3): the same position.
    for (size_t sl = 0; sl < plan.baryons.size(); ++sl) {
        const int b = plan.baryons[sl], partner = iso_partner(b);
        plan.slot_partner_iso.push_back(partner >= 0 ? slot_of[partner] : (int)sl);
        plan.slot_sign_iso.push_back(partner >= 0 && b != NBS_SIGMA_M ? -1 : +1);
    }

    // ---- program of the pipelined kernel (nbs_tables.hpp): simulate the walk over one task, full chain at q then
    // half chain at -q, with four block slots; repeat from the end state until the assignment is periodic.
    {
        struct Need { int id, nslots; }; // id = block slot * 2 + (1 if taken at -q)
        const int n = plan.chain_full_n + plan.chain_half_n;
        auto need_of = [&](int i, int side) {
            const ChainRec& cr = plan.chain[i];
            const Pair3Rec& pr = plan.pairs3[cr.pair];
            const bool neg = i >= plan.chain_full_n; // half chain: the item's momentum is -q
            const int slot = side ? pr.slot2 : pr.slot1;
            const int at_minus = (side == 1) != neg;  // B~1 at the item's momentum, B~2 at minus that
            return Need{slot * 2 + (at_minus ? 1 : 0), plan.slot_kind[slot] == BK_FULL ? 2 : 1};
        };
        struct SlotState { int id = -1, last = -(1 << 20); };
        struct Sched { std::vector<CItem> items; std::vector<std::vector<CLoad>> rel; bool ok = true; };
        auto simulate = [&](std::array<SlotState, C_NSLOT>& st, bool drain) {
            Sched sc;
            sc.items.resize(n);
            sc.rel.assign(n, {});
            for (auto& x : st) x.id = -1; // blocks of the previous task are never reused (another momentum)
            if (drain) for (auto& x : st) x.last = -1; // every slot is free when the last item of the previous task is complete
            for (int i = 0; i < n; ++i) {
                const ChainRec& cr = plan.chain[i];
                CItem& it = sc.items[i];
                it.pair = cr.pair; it.nunits = cr.nunits; it.unit_begin = cr.unit_begin; it.ndiags = cr.ndiags;
                it.diag_begin = cr.diag_begin;
                it.flags = (i >= plan.chain_full_n) ? 64 : 0;
                it.rel_begin = it.rel_end = 0;
                int base[2] = {-1, -1};
                bool fresh[2] = {false, false};
                const Need nd[2] = {need_of(i, 0), need_of(i, 1)};
                for (int side = 0; side < 2; ++side) // resident blocks first
                    for (int s = 0; s < C_NSLOT; ++s)
                        if (base[side] < 0 && st[s].id == nd[side].id && (s == 0 || st[s - 1].id != nd[side].id)) base[side] = s;
                for (int side = 0; side < 2; ++side) {
                    if (base[side] >= 0) continue;
                    const int other = 1 - side;
                    auto taken = [&](int s) { // slot s belongs to the other block of this item
                        return base[other] >= 0 && s >= base[other] && s < base[other] + nd[other].nslots;
                    };
                    int best = -1, best_last = 1 << 30;
                    for (int s = 0; s + nd[side].nslots <= C_NSLOT; s += nd[side].nslots) {
                        bool free_ok = true;
                        int last = -(1 << 20);
                        for (int k = s; k < s + nd[side].nslots; ++k) { free_ok = free_ok && !taken(k); last = std::max(last, st[k].last); }
                        // an antisymmetric block prefers a slot whose neighbour is busy as well (keeps pairs of slots free for full blocks)
                        if (free_ok && last < best_last) { best = s; best_last = last; }
                    }
                    if (best < 0 || best_last >= i) { sc.ok = false; return sc; }
                    base[side] = best; fresh[side] = true;
                    CLoad ld;
                    ld.src = (nd[side].id >> 1) | ((nd[side].id & 1) << 8);
                    ld.dst = c_slot_base(best);
                    ld.bytes = (uint32_t)block_elems(plan.slot_kind[nd[side].id >> 1]) * 16u;
                    ld.bar = best;
                    int dep = best_last; // the item whose completion frees the destination; < 0: an item of the previous task
                    if (dep < -n) dep = -n; // free from the start: issue with the first item of the previous task
                    if (dep < 0) { ld.src |= 1 << 9; sc.rel[dep + n].push_back(ld); }
                    else sc.rel[dep].push_back(ld);
                    for (int k = best; k < best + nd[side].nslots; ++k) st[k].id = -1; // whatever lived there is overwritten
                    st[best].id = nd[side].id;
                    if (nd[side].nslots == 2) st[best + 1].id = nd[side].id;
                }
                for (int side = 0; side < 2; ++side)
                    for (int k = base[side]; k < base[side] + nd[side].nslots; ++k) st[k].last = i;
                it.off1 = c_slot_base(base[0]); it.off2 = c_slot_base(base[1]);
                it.ps1 = (uint32_t)plane_elems(plan.slot_kind[nd[0].id >> 1]) * 16u;
                it.ps2 = (uint32_t)plane_elems(plan.slot_kind[nd[1].id >> 1]) * 16u;
                if (fresh[0]) it.flags |= 1 + base[0];
                if (fresh[1]) it.flags |= (1 + base[1]) << 3;
            }
            for (auto& x : st) x.last -= n; // relative to the next task
            return sc;
        };
        auto same = [](const Sched& a, const Sched& b) {
            if (a.items.size() != b.items.size()) return false;
            for (size_t i = 0; i < a.items.size(); ++i) {
                if (a.items[i].off1 != b.items[i].off1 || a.items[i].off2 != b.items[i].off2 || a.items[i].flags != b.items[i].flags) return false;
                if (a.rel[i].size() != b.rel[i].size()) return false;
                for (size_t j = 0; j < a.rel[i].size(); ++j)
                    if (a.rel[i][j].src != b.rel[i][j].src || a.rel[i][j].dst != b.rel[i][j].dst) return false;
            }
            return true;
        };
        plan.cprog_ok = false;
        if (n >= C_NREC) {
            std::array<SlotState, C_NSLOT> st;
            Sched prev, cur;
            bool periodic = false;
            for (int iter = 0; iter < 8 && !periodic; ++iter) {
                cur = simulate(st, false);
                if (!cur.ok) break;
                periodic = iter > 0 && same(prev, cur);
                prev = cur;
            }
            if (!periodic) {
                std::array<SlotState, C_NSLOT> st2;
                cur = simulate(st2, true);
                plan.cprog_drain = 1;
            }
            if (cur.ok) {
                for (int i = 0; i < n; ++i) {
                    cur.items[i].rel_begin = (int)plan.cloads.size();
                    for (auto& ld : cur.rel[i]) plan.cloads.push_back(ld);
                    cur.items[i].rel_end = (int)plan.cloads.size();
                }
                plan.cprog = cur.items;
                plan.cprog_ok = true;
            }
        }
    }

    // tile-wise plan: expansion map of a two-plane chunk of an antisymmetric block
    for (int kind = BK_ASYM13; kind <= BK_ASYM23; ++kind) {
        std::vector<int>& g = plan.gather_pp[kind - 1];
        g.assign(2 * SM_PLANE, -1);
        for (int al = 0; al < 2; ++al)
            for (int x1 = 0; x1 < NXI; ++x1)
                for (int x2 = 0; x2 < NXI; ++x2)
                    for (int x3 = 0; x3 < NXI; ++x3) {
                        if ((kind == BK_ASYM13 ? x1 : x2) == x3) continue; // diagonal: zero
                        const Located loc = locate(kind, x1, x2, x3);
                        g[al * SM_PLANE + sm_index(x1, x2, x3)] = (al * AS_PLANE + loc.idx) | (loc.sign < 0 ? (1 << 30) : 0);
                    }
    }
    return "";
}

} // namespace nbs
