// Host table generator (row a0 of DESIGN.md): the paper's CPU-side "diagramatical classification"
// whose Structure-of-Arrays result is copied to the device before the kernels run
// (PAPER.md:108, :115).  Pure host C++, no CUDA; shares no code with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/nbs.h"

namespace nbs {

constexpr int NXI = 12;           // colour x spin
constexpr int NTRIPLE = 1728;     // 12^3 source index triples of a normal block
constexpr int BLOCK_ELEMS = 6912; // 4 sink spins x 12^3

// Shared-memory layout of one sink-spin plane of a normal block in the product kernel: the source
// triple (xi1, xi2, xi3) sits at xi1*145 + xi2*12 + (xi3 + xi2) mod 12.  With this skew four
// consecutive values of any one xi fall into four different 16-byte bank groups modulo 4, and the
// plane stride 1740 = 4 (mod 8) puts two adjacent planes into the two halves of the 8 bank groups:
// the 8 lanes of a quarter warp (2 planes x 4 consecutive k) then gather without bank conflicts.
constexpr int SM_STRIDE1 = 145;
constexpr int SM_PLANE = 12 * SM_STRIDE1;  // 1740
constexpr int SM_BLOCK = 4 * SM_PLANE;     // 6960 complex per staged block
#ifdef __CUDACC__
#define NBS_HD __host__ __device__
#else
#define NBS_HD
#endif
NBS_HD constexpr int sm_index(int xi1, int xi2, int xi3) { return xi1 * SM_STRIDE1 + xi2 * 12 + (xi3 + xi2) % 12; }

// Blocks of baryons with two quarks of one flavour are antisymmetric under the exchange of those
// two source slots (the Wick sign of exchanging the two identical quark fields): p, Sigma+, Sigma-
// in slots (1,3), n, Xi0, Xi- in slots (2,3).  Only the entries with xi_a < xi_b are built, Fourier
// transformed and staged by the product kernel (66 of 144 index pairs), in the "compact" layout
//   antisymmetric plane: [xi_c (free slot): 12][72 positions] + 4 pads = 868 entries,
//   the pair (xi_a < xi_b) of row xi_c at position (as_pair_pos(xi_a, xi_b) + xi_c) mod 72,
// where as_pair_pos = 4 m + (xi_a + xi_b) mod 4 with m a running number inside the residue class.  The position
// is therefore congruent to xi_a + xi_b + xi_c modulo 4 -- the same rule as sm_index -- and the plane stride
// 868 = 4 (mod 8): every gather pattern that is free of bank conflicts on a full staged block is free of them on
// the compact block too, mirrored entries included (the sum is symmetric in xi_a, xi_b).  The six unused
// positions of a row (52, 54, 60, 62, 68, 70 before the rotation) and the plane pads are zero; the identically
// vanishing diagonal xi_a == xi_b is read from the unused position of the matching residue.
enum { BK_FULL = 0, BK_ASYM13 = 1, BK_ASYM23 = 2 };
constexpr int AS_ROW = 72;
constexpr int AS_PLANE = 12 * AS_ROW + 4; // 868
constexpr int AS_BLOCK = 4 * AS_PLANE;    // 3472 complex per compact antisymmetric block
constexpr int AS_ROW_PADS = 6;
NBS_HD constexpr int as_pad_pos(int i) { return 52 + 8 * (i >> 1) + 2 * (i & 1); } // 52, 54, 60, 62, 68, 70
NBS_HD constexpr int as_pair_pos(int a, int b) { // a < b
    const int a0 = a & 3, a1 = a >> 2, b1 = b >> 2, rho = (a + b) & 3;
    const int m = (a1 < b1) ? a0 + 4 * (a1 + b1 - 1) : 12 + 2 * a1 + ((a0 >> 1) | (a0 & (rho >> 1)));
    return 4 * m + rho;
}
NBS_HD constexpr int as_index(int a, int b, int c) { return c * AS_ROW + (as_pair_pos(a, b) + c) % AS_ROW; } // a < b
NBS_HD constexpr int as_zero_index(int a, int c) { return c * AS_ROW + (52 + ((2 * a) & 3) + c) % AS_ROW; } // a == b
NBS_HD constexpr int plane_elems(int kind) { return kind == BK_FULL ? SM_PLANE : AS_PLANE; }
NBS_HD constexpr int block_elems(int kind) { return 4 * plane_elems(kind); }
struct Located {
    int idx;  // position inside the sink-spin plane of the compact layout
    int sign; // +1, or -1 if the stored partner carries the opposite sign; 0: identically zero (idx = a zero pad)
};
NBS_HD constexpr Located locate(int kind, int xi1, int xi2, int xi3) {
    if (kind == BK_FULL) return Located{sm_index(xi1, xi2, xi3), 1};
    const int a = (kind == BK_ASYM13) ? xi1 : xi2, b = xi3, c = (kind == BK_ASYM13) ? xi2 : xi1;
    if (a == b) return Located{as_zero_index(a, c), 0};
    if (a < b) return Located{as_index(a, b, c), 1};
    return Located{as_index(b, a, c), -1};
}
int block_kind(int baryon); // from the slot flavours of eqs. 2.2-2.3

// One elementary operator  eps_abc (q_f0,a  C g5  q_f1,b) q_f2,c  with a real coefficient
// (eqs. 2.2-2.3).  Flavours: 0 = u, 1 = d, 2 = s.
struct ElemTerm {
    double coef;
    int f[3];
};
struct BaryonDef {
    int slot[3]; // flavour of the three source quarks the block is contracted with (eq. 2.5)
    int nterm;
    ElemTerm term[3];
};
const BaryonDef& baryon_def(int id);

// One term of a normal block (eq. 2.5):
//   out[a][xi0,xi1,xi2] += coef * sum_c D^{f0 f1}_c(xi_{perm0}, xi_{perm1}) S_{f2}[(c,a), xi_{perm2}]
struct BlockTerm {
    double coef;
    int f0, f1, f2;
    int perm[3];
};
std::vector<BlockTerm> block_terms(int baryon);

// ---- product kernel (DMMA) records ----------------------------------------------------------
// A "unit" is the work of one warp: a few diagrams (or k-ranges of one diagram) of ONE elementary
// correlator that share one accumulator layout (class).  Classes (which effective
// block carries a3 / a4):
//   0: 16x16, B~1 carries a3, B~2 carries a4      1: 16x16, B~1 carries a4, B~2 carries a3
//   2: 64x4,  B~1 carries a3 and a4               3: 4x64,  B~2 carries a3 and a4
//
// Gather tables: one uint2 {off_plus, off_minus} per PAIR of gather terms of an effective-block
// entry (eq. 4.2): entry = sum_j ( blk[off_plus_j] - blk[off_minus_j] ).  Every entry has as many
// +1 as -1 terms (the eps (C g5) weights are balanced, and sigma_P only swaps the two halves), so no
// sign bits are needed; a padded k (k >= K) has off_plus == off_minus and contributes exactly 0.
// Offsets are BYTE offsets into the staged block of that side, with the sink-spin plane of the
// reading lane folded in (the kernel adds compile-time plane offsets only):
//   16x16 sides    [k][row r = 2*c + (a & 1)][nw]          planes a = (r & 1) + {0, 2}
//   64x4  A side   [k][row r = 2*(cX & 3) + (a & 1)][g = cX >> 2][1]   planes a = (r & 1) + {0, 2}
//   64x4  B side   [k][a][nw]                               plane a
// k is padded to a multiple of 4 (one DMMA k-step).
constexpr int MAX_PAIR_ELEMS = 16;
constexpr int MAX_PAIR_UNITS = 128; // unit and diagram records of one sink pair are staged in shared memory
constexpr int MAX_PAIR_DIAGS = 192;
struct Diag3Rec {
    uint32_t offA, offB; // uint2 offsets into Plan::tab3: operand A (the M side) and operand B (the N side)
    uint16_t sbeg, send; // k-steps [sbeg, send) of this diagram covered by this record
    uint8_t nwA, nwB;    // uint2 words (term pairs) per entry
    uint16_t K;          // size of the shared index (1, 9, 36, 144)
};
struct Unit3Rec {        // in schedule order (cost descending) per sink pair
    int diag_begin, diag_end; // range in the sink pair's diagram records (relative to Pair3Rec::diag_begin)
    int cls;
    int slot;                 // row of the per-item unit scratch (units grouped by elementary correlator)
};
struct Pair3Rec {
    int slot1, slot2;
    int unit_begin, nunits;  // Plan::units3 range (schedule order)
    int diag_begin, ndiags;  // Plan::diags3 range
    int nelem;
    int elem_unit_begin[MAX_PAIR_ELEMS + 1]; // scratch-row ranges per elementary correlator
    int chan_begin, nchan;   // range in Plan::pair_chans
    int swap_mask;           // bit e: some channel needs elementary correlator e with a3 <-> a4 exchanged
    int self_swap;           // 1: identical sink baryons; 2: a field and its u <-> d image (reduced plan of the isospin limit);
                             // computed for q <= -q only, mirrored to -q by the epilogue (PairChanRec::mirror_*)
};
struct PairChanRec {
    int ch, local; // channel index; position of the channel among the channels of its sink pair (row of the tile-wise plan's Ft)
    // isospin limit, reduced channel list (IsoRelation): a second channel that the epilogue writes from this one,
    // F[alias_ch] = alias_sign * F[ch], with the source spins a3 <-> a4 exchanged if alias_swap; alias_ch = -1: none
    int alias_ch, alias_swap;
    double alias_sign;
    // what the epilogue writes at -q for a pair that is computed for the momenta q <= -q only (Pair3Rec::self_swap):
    // F[mirror_ch](-q)_{a2 a1 ..} = mirror_sign * F[ch](q)_{a1 a2 ..}, with a3 <-> a4 exchanged as well if mirror_swap.
    // Identical sink baryons (reading A11): the channel itself, sign -1.  Isospin limit, sink pair (B, B') of a field
    // and its u <-> d image (p n, Sigma+ Sigma-, Xi- Xi0): the channel with the images of the source baryons.
    int mirror_ch, mirror_swap;
    double mirror_sign;
    double coef[MAX_PAIR_ELEMS];  // channel = sum_e coef[e] * E_e + coefS[e] * (E_e with a3 <-> a4), eqs. 2.2-2.3;
    double coefS[MAX_PAIR_ELEMS]; // coefS carries the minus sign of the source swap (reading A11)
};
struct ChainRec { // order in which one CTA walks the sink pairs of one momentum; self-contained staging descriptor
    int pair;
    int load1, load2; // 1: this item must (re)load B~1(q) / B~2(-q); 0: the staged block is reused
    int nunits;
    int unit_begin, ndiags, diag_begin, pad;
    int buf1, off1, buf2, off2; // Plan::slot_src of the two blocks
};

// ---- pipelined product kernel (k_product_c): compact antisymmetric blocks staged as they are -------------
// Shared memory holds four block slots: a compact antisymmetric block takes one, a full staged block two adjacent
// ones (0-1 or 2-3).  The slots are interleaved in units of half slots (C_HALF_BYTES = one full plane = two compact
// planes): slot s = 2 q + i owns the half slots 4 q + i and 4 q + i + 2, so that in BOTH kinds of block the sink-spin
// planes a and a + 2 lie C_PAIR_BYTES apart (a full block in slots 2 q, 2 q + 1 is simply contiguous): the gathers
// reach plane a + 2 through a compile-time offset.  One task = one momentum pair (q, -q): the full chain at q followed by
// the half chain at -q.  The host simulates the walk once (build_plan) and writes a static program: for every
// item the slots of its two blocks, which of them are fresh loads (the item waits for the slot's barrier), and
// a release list -- the bulk copies that may be issued as soon as the item is complete, because they overwrite
// blocks that nobody needs any more.  The program is cyclic: release lists near its end carry the first loads of
// the next task.
// Packed gather tables (Plan::tabc): one 32-bit word per (+, -) pair of gather terms, byte offsets inside ONE sink-spin
// plane of the block (the plane of the reading lane is part of its base pointer, so a table serves all planes):
//   bits 4-14 offset of the + term, bit 15 its flip flag, bits 20-30 offset of the - term, bit 31 its flip flag
//   (a set flip flag: the loaded value enters with the opposite sign -- compact blocks only, see build_plan).
//   16x16 sides  [k][c (carried spin)][nw]          64x4 A side  [k][cX & 3][g = cX >> 2]          64x4 B side  [k][nw = 4]
constexpr int C_TAB_LOOKAHEAD = 5; // k-steps the kernel's register pipeline may read past the end of a range (tables are padded by as many)
constexpr uint32_t C_HALF_BYTES = SM_PLANE * 16u;      // 27 840 >= 2 * AS_PLANE * 16 = 27 776
constexpr uint32_t C_PAIR_BYTES = 2u * C_HALF_BYTES;   // distance of the planes a and a + 2 of a staged block
constexpr int C_NSLOT = 4;
constexpr uint32_t C_BLOCKS_BYTES = 2u * C_NSLOT * C_HALF_BYTES; // 222 720
NBS_HD constexpr uint32_t c_slot_base(int s) { return (uint32_t)((s >> 1) * 4 + (s & 1)) * C_HALF_BYTES; }
constexpr int C_NREC = 3; // unit / diagram record buffers: a warp may run two items ahead of the slowest one
struct CItem { // 48 bytes, read as three int4
    int pair, nunits, unit_begin, ndiags;
    int diag_begin;
    uint32_t off1, off2;     // shared-memory byte offsets of B~1 and B~2 of this item (c_slot_base of their first slot)
    uint32_t ps1, ps2;       // bytes of one sink-spin plane of the two blocks (planes a, a + 1 are adjacent)
    int flags;               // bits 0-2: 1 + slot to wait for on side 1 (0: resident); bits 3-5: same for side 2;
                             // bit 6: the item belongs to momentum -q of the task (half chain)
    int rel_begin, rel_end;  // release list (Plan::cloads) of this item
};
struct CLoad { // 16 bytes
    int src;        // bits 0-7: block slot (Plan::baryons index); bit 8: at -q; bit 9: of the next task
    uint32_t dst;   // shared-memory byte offset
    uint32_t bytes;
    int bar;        // slot barrier that completes
};

struct uint2x { uint32_t x, y; }; // host mirror of CUDA uint2
struct int2x { int x, y; };

struct DiagramInfo { // host-side description (tests, statistics)
    int P[6];
    int sign;
    int K;
};

struct Plan {
    std::vector<nbs_channel> channels;
    std::vector<int> baryons; // needed sink baryon ids, slot order
    // compact site row (what k_blocks writes and the FFT transforms): every slot's block in the layout of its kind
    std::vector<int> slot_off, slot_kind;
    int row_elems = 0;
    // Antisymmetric slots are expanded after the FFT into a second buffer of full staged blocks
    // (row = n_asym * SM_BLOCK): expanded element j takes compact element gather[j] & 0x3fffffff of the
    // same site, negated if bit 30 is set; -1 = zero (pads and the diagonal xi_a == xi_b).
    std::vector<int> gather;
    int n_asym = 0;
    // where the product kernel stages slot s from: slot_src[s].x = 0: compact row at offset .y (full
    // kinds are already staged blocks there); 1: expanded row at offset .y
    std::vector<int2x> slot_src;
    // Isospin-limit fast path (used when the caller passes d == u): with identical u and d
    // propagators  n(xi1 xi2 xi3) = -p(xi2 xi1 xi3),  Sigma- = Sigma+,  Xi- = -Xi0  hold for the blocks, so the
    // derived slots (placed last in the compact row) are neither built nor transformed: n_slots_iso slots and
    // row_elems_iso components go through k_blocks / FFT, and gather_iso expands the derived ones from their partners.
    int n_slots_iso = 0, row_elems_iso = 0;
    std::vector<int> gather_iso;
    std::vector<int> chan_pair; // pair index of each channel
    double sumK_std = 0;        // sum over channels of sum_d K_d (the paper's count)
    double sumK_exec = 0;       // sum over the computed elementary correlators of pairs of different sink baryons
    double sumK_exec_self = 0;  // same for pairs of identical sink baryons (executed for about half of the momenta)
    // product kernel tables
    std::vector<Pair3Rec> pairs3;
    std::vector<Unit3Rec> units3;
    std::vector<Diag3Rec> diags3;
    std::vector<uint2x> tab3;
    std::vector<PairChanRec> pair_chans;
    std::vector<ChainRec> chain; // full chain, then the half chain, then one single-pair chain per sink pair
    int chain_full_n = 0, chain_half_n = 0;
    int chain_single_begin = 0; // chain[chain_single_begin + p]: sink pair p alone, both blocks loaded (tile-wise plan)
    // Tile-wise plan (configs[4], 96^3): a chunk holds two sink-spin planes of one baryon for all sites.  Expansion
    // map of a chunk of an antisymmetric block, [kind - 1][2 * SM_PLANE]: expanded element j takes compact element
    // gather_pp[j] & 0x3fffffff of the same site's compact plane pair [2][AS_PLANE], negated if bit 30 is set; -1 = zero.
    std::vector<int> gather_pp[2];
    int max_pair_units = 0;
    int max_pair_diags = 0;
    double sumKp_exec = 0; // executed k-steps x 4 (padding included)
    // pipelined kernel: packed gather tables in the layout of the block kind of each side (compact for
    // antisymmetric blocks), one diagram record per entry of diags3
    std::vector<uint32_t> tabc;
    std::vector<Diag3Rec> diagsc; // offA / offB in 32-bit words of tabc
    std::vector<CItem> cprog;   // one task: full chain at q, half chain at -q
    std::vector<CLoad> cloads;
    bool cprog_ok = false;      // false: the plan is too small / too large for the pipelined kernel
    int cprog_drain = 0;        // 1: no periodic slot assignment was found, every task starts from empty slots
    // isospin limit (d == u): derived slots are read from their partner's compact block with a sign
    std::vector<int> slot_partner_iso;  // [slot] slot to read (itself if not derived)
    std::vector<int> slot_sign_iso;     // [slot] +1 / -1
};

// Returns "" on success, else an error message (invalid id, flavour violation).
// iso_conj (reduced plan of the isospin limit only): per channel, 1 = this channel may not take part in a mirror relation
// (it carries a u <-> d image to write); a non-NULL vector switches the relation
//   F[B B' | B3 B4](q)_{a1 a2 a3 a4} = - eta_B eta_B' eta_3 eta_4 F[B B' | B3' B4'](-q)_{a2 a1 a3 a4}      (B' = image of B)
// on for every sink pair whose channel set is closed under it: such a pair is computed for q <= -q only.
// unit_split_steps: a diagram with more k-steps is split over several units; unit_cost_max: diagrams are packed into a
// unit up to this cost (2 per 16x16 k-step, 3 per 64x4 k-step).  Defaults: whole diagrams (K = 144 has 36 k-steps),
// measured best with 12 compute warps: (36, 120 - 160) 58.8 ms, (18, 80) 60.1, (18, 240) 61.4, (36, 200) 60.8 at 32^3.
constexpr int UNIT_SPLIT_STEPS_DEFAULT = 36, UNIT_COST_MAX_DEFAULT = 140;
std::string build_plan(const std::vector<nbs_channel>& channels, Plan& plan, int unit_split_steps = UNIT_SPLIT_STEPS_DEFAULT,
                       int unit_cost_max = UNIT_COST_MAX_DEFAULT, const std::vector<char>* iso_conj = nullptr);

// Channel relations of the isospin limit (u and d propagators identical): relabelling u <-> d maps every
// interpolating field of eqs. 2.2-2.3 to +-1 times another one (p <-> n, Sigma+ <-> Sigma-, Xi0 <-> -Xi-, Lambda -> -Lambda,
// Sigma0 -> Sigma0, X_u <-> -X_d, X_s -> -X_s) and leaves the path integral unchanged, so
//   <B1 B2 | B3 B4> = eta1 eta2 eta3 eta4 <B1' B2' | B3' B4'>,   and   <.. | B4' B3'>_{a3 a4} = - <.. | B3' B4'>_{a4 a3}.
// rel[i].from = -1: channel i is computed; else channel i = sign * channel `from` (a3 <-> a4 exchanged if swap34),
// `from` < i and itself computed.  The signs come from the operator table (baryon_iso_mirror), not from a list.
struct IsoRelation { int from, sign, swap34; };
std::vector<IsoRelation> iso_channel_relations(const std::vector<nbs_channel>& channels);
// u <-> d image of an interpolating field: returns the field id and writes eta = +-1; -1 if the image is no field of the table
int baryon_iso_mirror(int baryon, int* eta);

// Diagrams of one channel in enumeration order (source terms major, permutations lexicographic).
std::string channel_diagrams(const nbs_channel& ch, std::vector<DiagramInfo>& out);

std::vector<nbs_channel> standard_channels();

} // namespace nbs
