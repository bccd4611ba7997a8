// (ii)+(iii) EffectiveBaryonBlocks fused into MultiplicationEffectiveBlocks, eqs. 4.2-4.3
// (PAPER.md:104-115), on the FP64 tensor path (DMMA.8x8x4, the native FP64 MMA of sm_100a).
//
// Per diagram d the sum over the shared index xi~_d is a small complex GEMM (eq. 4.3)
//     out[m][n] += sum_k  eff1[m][k] * eff2[n][k],   m = (a1, carried spins), n = (a2, carried spins)
// of shape 16 x 16 x K or 64 x 4 x K (K = 1, 9, 36, 144).  One warp owns a "unit"
// (a few diagrams, or a k-range of one): every effective-block entry (eq. 4.2: a difference of two
// sums of 1, 4 or 12 normal-block entries) is gathered from shared memory exactly once, straight
// into the lane that holds it as an MMA fragment, and is then used by 8 output columns through the
// tensor path.  The effective blocks never exist in memory.
//
// Persistent, warp-specialised kernel, one CTA per SM:
//   * 10 compute warps.  A CTA takes a momentum q from a global counter and walks the sink pairs in
//     "chain" order (consecutive pairs share B~1(q) or B~2(-q), so only ~15 instead of 28 blocks
//     are staged per q).  The q-space normal blocks are stored in HBM in exactly the padded,
//     bank-conflict-free layout the gathers want, so staging is one thread issuing bulk
//     asynchronous copies (cp.async.bulk, completion on an mbarrier).  Warps take units from a
//     shared-memory counter, accumulate in registers and write each unit's 256 spin components to
//     a double-buffered per-CTA scratch.
//   * 2 epilogue warps.  While the compute warps work on item i+1 they sum the unit results of
//     item i per elementary correlator in a fixed order (bitwise reproducible) and write the
//     channel correlators (coefficients of eqs. 2.2-2.3).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstddef>

#include "nbs_tables.hpp"

namespace nbs {

constexpr int PROD_CWARPS = 10, PROD_EWARPS = 2;
constexpr int PROD_CTHREADS = PROD_CWARPS * 32, PROD_ETHREADS = PROD_EWARPS * 32;
constexpr int PROD_THREADS = PROD_CTHREADS + PROD_ETHREADS;
constexpr uint32_t PLANE_BYTES = SM_PLANE * 16u;  // 27 840
constexpr uint32_t BLOCK_BYTES = SM_BLOCK * 16u;  // 111 360
// osign of combine_item: only the pipelined kernel (nbs_product_c.cuh) passes a value other than 1.
// shared-memory map (bytes)
constexpr uint32_t SMO_S1 = 0, SMO_S2 = BLOCK_BYTES, SMO_UNITS = 2 * BLOCK_BYTES;
constexpr uint32_t SMO_DIAGS = SMO_UNITS + MAX_PAIR_UNITS * 16u;
constexpr int EPI_CG = 6; // channels per epilogue pass over the unit results
constexpr uint32_t SMO_EPI = SMO_DIAGS + MAX_PAIR_DIAGS * 16u; // epilogue's copy of the pair and channel records
constexpr uint32_t EPI_PAIR_BYTES = (sizeof(Pair3Rec) + 15u) / 16u * 16u;
constexpr uint32_t SMO_CTRL = SMO_EPI + EPI_PAIR_BYTES + EPI_CG * (uint32_t)sizeof(PairChanRec) + 8u;
constexpr int PROD_NBUF = 4; // depth of the unit-result ring between compute and epilogue warps
constexpr size_t PROD_SMEM = SMO_CTRL + 128;
static_assert(sizeof(Unit3Rec) == 16 && sizeof(Diag3Rec) == 16 && sizeof(ChainRec) == 48, "record sizes");
static_assert(PROD_SMEM <= 232448, "shared memory budget of one SM");

struct ProdCtrl { // at SMO_CTRL
    unsigned long long mbar1, mbar2; // completion of the bulk copies into s1 / s2
    int next_unit;                   // work counter of the current item
    int pad;
    long long qtask[2];              // prefetched momentum-task indices (alternating slots)
    int meta_q[PROD_NBUF], meta_pair[PROD_NBUF]; // item descriptors handed to the epilogue warps
    int meta_acc[PROD_NBUF];                     // direct mode: add to the result already stored for this r
};

// ---- PTX helpers ----------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ double dneg(double v) {
    return __hiloint2double(__double2hiint(v) ^ (int)0x80000000u, __double2loint(v));
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, uint32_t parity) {
    const uint32_t a = smem_u32(bar);
    uint32_t ok = 0;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, void* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void named_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void named_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
enum { BAR_COMPUTE = 1, BAR_FULL0 = 2, BAR_EMPTY0 = 2 + PROD_NBUF, BAR_EPI = 2 + 2 * PROD_NBUF };
static_assert(3 + 2 * PROD_NBUF <= 16, "named barriers");
static_assert(sizeof(Pair3Rec) % 4 == 0 && sizeof(PairChanRec) % 8 == 0 && SMO_CTRL % 8 == 0, "record alignment");

__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
__device__ __forceinline__ void bulk_prefetch_l2(const void* p, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// ---- gathers (eq. 4.2) ----------------------------------------------------------------------
// One table word = one (+, -) pair of byte offsets into a staged block.  ld_pair issues the
// shared-memory loads for NP sink-spin planes (plane stride PS bytes), sub_pair folds them.
template <int NP, uint32_t PS>
__device__ __forceinline__ void ld_pair(const char* __restrict__ blk, uint2 w, double2 (&u)[NP], double2 (&v)[NP]) {
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        u[p] = *reinterpret_cast<const double2*>(blk + w.x + p * PS);
        v[p] = *reinterpret_cast<const double2*>(blk + w.y + p * PS);
    }
}
template <int NP, bool FIRST>
__device__ __forceinline__ void sub_pair(const double2 (&u)[NP], const double2 (&v)[NP], double2 (&out)[NP]) {
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        if (FIRST) out[p] = make_double2(u[p].x - v[p].x, u[p].y - v[p].y);
        else { out[p].x += u[p].x - v[p].x; out[p].y += u[p].y - v[p].y; }
    }
}

// ---- classes 0, 1: 16 x 16 outputs -----------------------------------------------------------
// MMA row = 2*c1 + (a1 & 1) in tile i = a1 >> 1 (from B~1), MMA column likewise from B~2; lane =
// 4*row + k.  The 8 lanes of a quarter warp are 2 adjacent planes x 4 consecutive k: no conflicts.
// Complex products with three real multiplications (Gauss): with P1 = sum Ar Br, P2 = sum Ai Bi and
// P3 = sum (Ar + Ai)(Br + Bi), Re = P1 - P2 and Im = P3 - P1 - P2.  12 DMMAs per k-step instead of 16
// for 4 more FP64 adds: the FP64 units (shared by DMMA and DADD) do 13 % less per k-step.
// NT = MMA tiles per side: 2 (whole blocks staged: a1, a2 = 0..3) or 1 (tile-wise plan: one plane pair per side).
template <int NT>
struct AccSquare {
    double p1[NT][NT][2], p2[NT][NT][2], p3[NT][NT][2];
};
template <int NT>
__device__ __forceinline__ void mma_square(AccSquare<NT>& c, const double2 (&A)[NT], const double2 (&B)[NT]) {
    double sA[NT], sB[NT];
#pragma unroll
    for (int i = 0; i < NT; ++i) { sA[i] = A[i].x + A[i].y; sB[i] = B[i].x + B[i].y; }
#pragma unroll
    for (int i = 0; i < NT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            dmma884(c.p1[i][j][0], c.p1[i][j][1], A[i].x, B[j].x);
            dmma884(c.p2[i][j][0], c.p2[i][j][1], A[i].y, B[j].y);
            dmma884(c.p3[i][j][0], c.p3[i][j][1], sA[i], sB[j]);
        }
}

__device__ __forceinline__ Diag3Rec load_diag(const Diag3Rec* p) { // p: shared memory
    const int4 v = *reinterpret_cast<const int4*>(p);
    Diag3Rec d;
    d.offA = (uint32_t)v.x; d.offB = (uint32_t)v.y;
    d.sbeg = (uint16_t)((uint32_t)v.z & 0xffffu); d.send = (uint16_t)((uint32_t)v.z >> 16);
    d.nwA = (uint8_t)((uint32_t)v.w & 0xffu); d.nwB = (uint8_t)(((uint32_t)v.w >> 8) & 0xffu);
    d.K = (uint16_t)((uint32_t)v.w >> 16);
    return d;
}

template <bool TILE>
__device__ __forceinline__ void run_unit_square(const Unit3Rec u, const Diag3Rec* diags,
                                                const uint2* __restrict__ tab, const char* s1, const char* s2,
                                                double2* __restrict__ out, int lane, int ti, int tj) {
    const int r = lane >> 2, kk = lane & 3;
    constexpr uint32_t PS = 2 * PLANE_BYTES;
    constexpr int NT = TILE ? 1 : 2;
    AccSquare<NT> acc = {};
    for (int d = u.diag_begin; d < u.diag_end; ++d) {
        const Diag3Rec dr = load_diag(diags + d);
        const int nsteps = dr.send - dr.sbeg;
        if (dr.nwA == 1) {
            // software pipeline: table words two k-steps ahead, shared-memory gathers one ahead
            const uint2* tA = tab + dr.offA + (dr.sbeg * 4 + kk) * 8 + r;
            const uint2* tB = tab + dr.offB + (dr.sbeg * 4 + kk) * 8 + r;
            uint2 wa = __ldg(tA), wb = __ldg(tB);
            uint2 na = __ldg(tA + 32), nb = __ldg(tB + 32);
            double2 A[NT], B[NT], ua[NT], va[NT], ub[NT], vb[NT];
            ld_pair<NT, PS>(s1, wa, ua, va);
            ld_pair<NT, PS>(s2, wb, ub, vb);
            sub_pair<NT, true>(ua, va, A);
            sub_pair<NT, true>(ub, vb, B);
            for (int s = 0; s < nsteps; ++s) {
                tA += 32; tB += 32;
                wa = na; wb = nb;
                ld_pair<NT, PS>(s1, wa, ua, va); // one step past the end reads a valid (unused) entry
                ld_pair<NT, PS>(s2, wb, ub, vb);
                na = __ldg(tA + 32); nb = __ldg(tB + 32);
                prefetch_l1(tA + 5 * 32); prefetch_l1(tB + 5 * 32); // L2 latency > 2 k-steps: pull the words into L1 early
                mma_square(acc, A, B);
                sub_pair<NT, true>(ua, va, A);
                sub_pair<NT, true>(ub, vb, B);
            }
        } else {
            const int nw = dr.nwA; // == nwB (4 or 12 term pairs per entry)
            const uint2* tA = tab + dr.offA + ((dr.sbeg * 4 + kk) * 8 + r) * nw;
            const uint2* tB = tab + dr.offB + ((dr.sbeg * 4 + kk) * 8 + r) * nw;
            for (int s = 0; s < nsteps; ++s, tA += 32 * nw, tB += 32 * nw) {
                double2 A[NT], B[NT], ua[NT], va[NT], ub[NT], vb[NT];
                ld_pair<NT, PS>(s1, __ldg(tA), ua, va);
                ld_pair<NT, PS>(s2, __ldg(tB), ub, vb);
                sub_pair<NT, true>(ua, va, A);
                sub_pair<NT, true>(ub, vb, B);
                for (int j = 1; j < nw; ++j) {
                    ld_pair<NT, PS>(s1, __ldg(tA + j), ua, va);
                    ld_pair<NT, PS>(s2, __ldg(tB + j), ub, vb);
                    sub_pair<NT, false>(ua, va, A);
                    sub_pair<NT, false>(ub, vb, B);
                }
                mma_square(acc, A, B);
            }
        }
    }
#pragma unroll
    for (int i = 0; i < NT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int a1 = 2 * (TILE ? ti : i) + (r & 1), c1 = r >> 1;
                const int cc = 2 * kk + e, a2 = 2 * (TILE ? tj : j) + (cc & 1), c2 = cc >> 1;
                const int a3 = u.cls == 0 ? c1 : c2, a4 = u.cls == 0 ? c2 : c1;
                out[((a1 * 4 + a2) * 4 + a3) * 4 + a4] =
                    make_double2(acc.p1[i][j][e] - acc.p2[i][j][e], acc.p3[i][j][e] - acc.p1[i][j][e] - acc.p2[i][j][e]);
            }
}

// ---- classes 2, 3: 64 x 4 outputs ------------------------------------------------------------
// Operand A = the effective block that carries a3 and a4: row m = (aX, cX = a3*4 + a4); tile
// (j, g) holds aX in {2j, 2j+1}, cX in {4g .. 4g+3}; MMA row = 2*(cX & 3) + (aX & 1).  Operand B =
// the other effective block (n = aY).  The 8 MMA columns hold [Re | Im] of the 4 outputs:
//   C += Ar [Br | Bi];  C += Ai [-Bi | Br].
template <int NJ>
__device__ __forceinline__ void mma_wide(double (&acc)[NJ * 4][2], const double2 (&A)[4][NJ], double2 Bv, int hi) {
    const double b1 = hi ? Bv.y : Bv.x;
    const double b2 = hi ? Bv.x : dneg(Bv.y);
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
        for (int j = 0; j < NJ; ++j) dmma884(acc[j * 4 + g][0], acc[j * 4 + g][1], A[g][j].x, b1);
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
        for (int j = 0; j < NJ; ++j) dmma884(acc[j * 4 + g][0], acc[j * 4 + g][1], A[g][j].y, b2);
}

// Table words of one k-step of one lane: 4 A entries (g) and the 4 term pairs of the B entry.
template <int NJ>
__device__ __forceinline__ void wide_loads_A(const char* sA, uint4 a01, uint4 a23, double2 (&ua)[4][NJ], double2 (&va)[4][NJ]) {
    constexpr uint32_t PS = 2 * PLANE_BYTES;
    ld_pair<NJ, PS>(sA, make_uint2(a01.x, a01.y), ua[0], va[0]);
    ld_pair<NJ, PS>(sA, make_uint2(a01.z, a01.w), ua[1], va[1]);
    ld_pair<NJ, PS>(sA, make_uint2(a23.x, a23.y), ua[2], va[2]);
    ld_pair<NJ, PS>(sA, make_uint2(a23.z, a23.w), ua[3], va[3]);
}
// B entry (8 gather terms = 4 pairs): the lanes hi = 0 and hi = 1 of one (aY, k) need the same entry, so
// each gathers two of the four pairs and the halves are exchanged with a shuffle (lane ^ 16 flips hi):
// 8 instead of 14 FP64 adds and 4 instead of 8 shared-memory loads per k-step.
__device__ __forceinline__ void wide_loads_B(const char* sB, uint4 bw, double2 (&ub)[2][1], double2 (&vb)[2][1]) {
    ld_pair<1, 0>(sB, make_uint2(bw.x, bw.y), ub[0], vb[0]);
    ld_pair<1, 0>(sB, make_uint2(bw.z, bw.w), ub[1], vb[1]);
}
__device__ __forceinline__ void wide_fold_B(const double2 (&ub)[2][1], const double2 (&vb)[2][1], double2 (&Bv)[1]) {
    double2 part[1];
    sub_pair<1, true>(ub[0], vb[0], part);
    sub_pair<1, false>(ub[1], vb[1], part);
    const double ox = __shfl_xor_sync(0xffffffffu, part[0].x, 16), oy = __shfl_xor_sync(0xffffffffu, part[0].y, 16);
    Bv[0] = make_double2(part[0].x + ox, part[0].y + oy);
}

// Tile-wise plan (TILE): each side holds one plane pair.  The A side then has one MMA row tile per g (NJ = 1); the
// lanes of the B side with aY = 2, 3 gather from planes that are not staged, and their two output columns (columns
// of an MMA do not mix) are dropped at the flush.
template <bool TILE>
__device__ __forceinline__ void run_unit_wide(const Unit3Rec u, const Diag3Rec* diags,
                                              const uint2* __restrict__ tab, const char* s1, const char* s2,
                                              double2* __restrict__ out, int lane, int ti, int tj) {
    const int r = lane >> 2, kk = lane & 3, aY = r & 3, hi = r >> 2;
    const char* sA = (u.cls == 2) ? s1 : s2;
    const char* sB = (u.cls == 2) ? s2 : s1;
    constexpr int NJ = TILE ? 1 : 2;
    double acc[NJ * 4][2] = {};
    for (int d = u.diag_begin; d < u.diag_end; ++d) {
        const Diag3Rec dr = load_diag(diags + d); // nwA == 1, nwB == 4 (checked by the table generator)
        const int nsteps = dr.send - dr.sbeg;
        // A table [k][r][g] (4 uint2 = 2 uint4 per lane), B table [k][aY][4 pairs] (2 uint4 per lane)
        const uint4* tA = reinterpret_cast<const uint4*>(tab + dr.offA) + ((dr.sbeg * 4 + kk) * 8 + r) * 2;
        const uint4* tB = reinterpret_cast<const uint4*>(tab + dr.offB) + ((dr.sbeg * 4 + kk) * 4 + aY) * 2;
        // software pipeline: table words one k-step ahead; the A gathers of step s+1 fly under the
        // MMAs of step s, the (8-term) B gather of step s+1 is issued after them and folded at the
        // top of step s+1 (keeps the live registers under the 168 available per thread)
        double2 A[4][NJ], Bv[1], ua[4][NJ], va[4][NJ], ub[2][1], vb[2][1];
        wide_loads_A<NJ>(sA, __ldg(tA), __ldg(tA + 1), ua, va);
        wide_loads_B(sB, __ldg(tB + hi), ub, vb);
        uint4 na01 = __ldg(tA + 64), na23 = __ldg(tA + 65), nbw = __ldg(tB + 32 + hi);
#pragma unroll
        for (int g = 0; g < 4; ++g) sub_pair<NJ, true>(ua[g], va[g], A[g]);
        for (int s = 0; s < nsteps; ++s) {
            tA += 64; tB += 32;
            wide_fold_B(ub, vb, Bv);
            wide_loads_A<NJ>(sA, na01, na23, ua, va); // one step past the end reads valid (unused) entries
            na01 = __ldg(tA + 64); na23 = __ldg(tA + 65);
            prefetch_l1(tA + 3 * 64); prefetch_l1(tB + 3 * 32); // L2 latency > 1 k-step: pull the words into L1 early
            mma_wide<NJ>(acc, A, Bv[0], hi);
#pragma unroll
            for (int g = 0; g < 4; ++g) sub_pair<NJ, true>(ua[g], va[g], A[g]);
            wide_loads_B(sB, nbw, ub, vb);
            nbw = __ldg(tB + 32 + hi);
        }
    }
    double* o = reinterpret_cast<double*>(out);
    const int tX = (u.cls == 2) ? ti : tj, tY = (u.cls == 2) ? tj : ti; // plane pairs of the A and the B side
#pragma unroll
    for (int j = 0; j < NJ; ++j)
#pragma unroll
        for (int g = 0; g < 4; ++g)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int aX = 2 * (TILE ? tX : j) + (r & 1), cX = 4 * g + (r >> 1);
                const int cc = 2 * kk + e, part = cc >> 2;
                if (TILE && (cc & 3) >= 2) continue; // columns of the planes that are not staged
                const int ay = TILE ? 2 * tY + (cc & 3) : (cc & 3);
                const int a1 = u.cls == 2 ? aX : ay, a2 = u.cls == 2 ? ay : aX;
                o[2 * ((a1 * 4 + a2) * 16 + cX) + part] = acc[j * 4 + g][e];
            }
}

struct ProdArgs {
    // momentum-space normal blocks as full staged blocks: slot s is staged from buffer slot_src[s].x
    // (0: compact rows Bc[V][Rc], where the blocks without an antisymmetry are stored staged; 1: expanded
    // rows Be[V][Re] of the antisymmetric blocks) at complex offset slot_src[s].y inside the site row
    const double2* Bc;
    size_t Rc;
    const double2* Be;
    size_t Re;
    const int2* slot_src;
    int L;
    int chain_full_n, chain_half_n; // chain[0 .. full_n): all pairs (momenta q <= -q); then the half chain
    long long ntasks;    // momentum tasks = entries of qorder
    const int* qorder;   // [V] momenta with q and -q adjacent
    const Pair3Rec* pairs;
    const Unit3Rec* units;
    const Diag3Rec* diags;
    const uint2* tab;
    const PairChanRec* pair_chans;
    const ChainRec* chain; // [chain_full_n + chain_half_n]
    double2* scratch;    // [gridDim.x][PROD_NBUF][max_pair_units][256]
    int max_pair_units;
    double2* Ft;         // [V][nch_out][256]
    int ch_begin, nch_out;
    unsigned long long* counter; // zeroed before the launch
    // direct mode (tiny-L path, eq. 2.4 as a shifted sum): Bc / Be hold the x-space blocks, a task is
    // a displacement r, its items are (X, sink pair) with B1 at X + r and B2 at X, and Ft[r] accumulates over X
    int direct;
    // tile-wise plan (k_product_t<true>; BASELINE.json configs[4]): one sink pair per launch (chain[chain_base]),
    // sink spins a1 in {2 tile_i, 2 tile_i + 1}, a2 in {2 tile_j, 2 tile_j + 1}; B~1 / B~2 are staged from the
    // two-plane chunks c1[V][2 * SM_PLANE] / c2[V][2 * SM_PLANE]; Ft[q][channel of the pair (PairChanRec::local)][256].
    // For identical sink baryons the launch with tile_i != tile_j also writes the tile (tile_j, tile_i) by the
    // sink-swap relation (reading A11), at -q.
    const double2* c1;
    const double2* c2;
    int tile_i, tile_j, chain_base;
};

__device__ __forceinline__ size_t minus_q(int L, size_t q) {
    int x = (int)(q % L), y = (int)((q / L) % L), z = (int)(q / ((size_t)L * L));
    x = x ? L - x : 0; y = y ? L - y : 0; z = z ? L - z : 0;
    return x + (size_t)L * (y + (size_t)L * z);
}

__device__ __forceinline__ size_t shifted_site(int L, size_t X, size_t r) { // X + r, periodic
    const int x = (int)((X % L + r % L) % L), y = (int)(((X / L) % L + (r / L) % L) % L);
    const int z = (int)((X / ((size_t)L * L) + r / ((size_t)L * L)) % L);
    return x + (size_t)L * (y + (size_t)L * z);
}

// Epilogue of one item: elementary correlators = sums of unit results (fixed order), channel
// correlators = real combinations of them (eqs. 2.2-2.3) -> Ft[q][ch][256].  The pair record and
// the channel coefficients are first copied to shared memory (one L2 round trip for the item
// instead of one per use); thread et owns the spin components et + 64 m.
template <bool TILE>
__device__ __forceinline__ void combine_item(const ProdArgs& a, int ip, size_t q, bool accumulate,
                                             const double2* __restrict__ scr, int et, char* s_epi, double osign = 1.0) {
    Pair3Rec* pr = reinterpret_cast<Pair3Rec*>(s_epi);
    PairChanRec* pcs = reinterpret_cast<PairChanRec*>(s_epi + EPI_PAIR_BYTES);
    {
        const int* src = reinterpret_cast<const int*>(a.pairs + ip);
        if (et < (int)(sizeof(Pair3Rec) / 4)) reinterpret_cast<int*>(pr)[et] = __ldg(src + et);
    }
    named_sync(BAR_EPI, PROD_ETHREADS);
    const int nelem = pr->nelem, nchan = pr->nchan, swap_mask = pr->swap_mask;
    const size_t mq = minus_q(a.L, q);
    const bool mirror = !a.direct && pr->self_swap && (mq != q || (TILE && a.tile_i != a.tile_j));
    // Components of this thread.  Whole blocks: et + 64 m, m = a1 = 0..3 (et = a2 a3 a4).  Tile-wise plan: the launch
    // holds a1 in pair tile_i, a2 in pair tile_j, 64 components, one per thread (et = low bit of a1, low bit of a2, a3 a4).
    constexpr int NM = TILE ? 1 : 4;
    const int t_a1 = 2 * a.tile_i + (et >> 5), t_a2 = 2 * a.tile_j + ((et >> 4) & 1);
    auto comp = [&](int m) { return TILE ? (t_a1 * 4 + t_a2) * 16 + (et & 15) : et + 64 * m; };
    // sink swap: F~(-q)_{a2 a1 a3 a4} = - F~(q)_{a1 a2 a3 a4}
    auto mirror_comp = [&](int m) { return TILE ? (t_a2 * 4 + t_a1) * 16 + (et & 15) : ((et >> 4) * 4 + m) * 16 + (et & 15); };
    const int nrows = TILE ? nchan : a.nch_out;
    for (int c0 = 0; c0 < nchan; c0 += EPI_CG) {
        const int nc = min(EPI_CG, nchan - c0);
        {
            const double* src = reinterpret_cast<const double*>(a.pair_chans + pr->chan_begin + c0);
            const int nwords = nc * (int)(sizeof(PairChanRec) / 8);
            for (int i = et; i < nwords; i += PROD_ETHREADS) reinterpret_cast<double*>(pcs)[i] = __ldg(src + i);
        }
        named_sync(BAR_EPI, PROD_ETHREADS);
        double2 acc[EPI_CG][NM];
#pragma unroll
        for (int c = 0; c < EPI_CG; ++c)
#pragma unroll
            for (int m = 0; m < NM; ++m) acc[c][m] = make_double2(0.0, 0.0);
        for (int e = 0; e < nelem; ++e) {
            double2 s[NM];
#pragma unroll
            for (int m = 0; m < NM; ++m) s[m] = make_double2(0.0, 0.0);
            const int ub = pr->elem_unit_begin[e], ue = pr->elem_unit_begin[e + 1];
            // rows in groups of EG with all loads of a group in flight (an elementary correlator has
            // ~5 unit rows: a plain unrolled loop would run them one by one through its remainder)
            constexpr int EG = 4;
            for (int ul = ub; ul < ue; ul += EG) {
                double2 v[EG][NM];
#pragma unroll
                for (int j = 0; j < EG; ++j)
#pragma unroll
                    for (int m = 0; m < NM; ++m)
                        v[j][m] = (ul + j < ue) ? __ldcg(scr + (size_t)(ul + j) * 256 + comp(m)) : make_double2(0.0, 0.0);
#pragma unroll
                for (int j = 0; j < EG; ++j)
#pragma unroll
                    for (int m = 0; m < NM; ++m) {
                        s[m].x += v[j][m].x;
                        s[m].y += v[j][m].y;
                    }
            }
            // source swap (reading A11): the same sums at the component with a3 <-> a4
            // exchanged live in another lane of the same 16-lane group
            const bool sw = (swap_mask >> e) & 1;
            double2 ss[NM];
            if (sw) {
                const int src_lane = (et & 0x10) | ((et & 3) << 2) | ((et >> 2) & 3);
#pragma unroll
                for (int m = 0; m < NM; ++m) {
                    ss[m].x = __shfl_sync(0xffffffffu, s[m].x, src_lane);
                    ss[m].y = __shfl_sync(0xffffffffu, s[m].y, src_lane);
                }
            }
#pragma unroll
            for (int c = 0; c < EPI_CG; ++c) {
                if (c < nc) {
                    const double k = pcs[c].coef[e];
#pragma unroll
                    for (int m = 0; m < NM; ++m) {
                        acc[c][m].x = fma(k, s[m].x, acc[c][m].x);
                        acc[c][m].y = fma(k, s[m].y, acc[c][m].y);
                    }
                    if (sw) {
                        const double ks = pcs[c].coefS[e];
#pragma unroll
                        for (int m = 0; m < NM; ++m) {
                            acc[c][m].x = fma(ks, ss[m].x, acc[c][m].x);
                            acc[c][m].y = fma(ks, ss[m].y, acc[c][m].y);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int c = 0; c < EPI_CG; ++c) {
            if (c < nc) {
                const int ch = TILE ? pcs[c].local : pcs[c].ch - a.ch_begin;
                if (ch >= 0 && ch < nrows) {
#pragma unroll
                    for (int m = 0; m < NM; ++m) { acc[c][m].x *= osign; acc[c][m].y *= osign; } // +-1 (isospin limit: sign of a derived block)
                    if (accumulate) { // direct mode, X > 0: the same thread wrote this entry for the previous X
#pragma unroll
                        for (int m = 0; m < NM; ++m) {
                            const double2 old = __ldcg(a.Ft + (q * nrows + ch) * 256 + comp(m));
                            acc[c][m].x += old.x;
                            acc[c][m].y += old.y;
                        }
                    }
#pragma unroll
                    for (int m = 0; m < NM; ++m) __stcs(a.Ft + (q * nrows + ch) * 256 + comp(m), acc[c][m]);
                    if (mirror) {
#pragma unroll
                        for (int m = 0; m < NM; ++m)
                            __stcs(a.Ft + (mq * nrows + ch) * 256 + mirror_comp(m), make_double2(-acc[c][m].x, -acc[c][m].y));
                    }
                }
            }
        }
        named_sync(BAR_EPI, PROD_ETHREADS); // the channel records may be overwritten by the next pass / item
    }
}

// L1 prefetch of the head (8 lines each) of the two gather tables of a unit's first diagram record.
__device__ __forceinline__ void prefetch_unit(const Unit3Rec* urec, const Diag3Rec* drecs, const uint2* __restrict__ tab,
                                              int lane) {
    if (lane < 16) {
        const int4 uv = *reinterpret_cast<const int4*>(urec);
        const int4 dv = *reinterpret_cast<const int4*>(drecs + uv.x);
        const uint32_t sbeg = (uint32_t)dv.z & 0xffffu, nwA = (uint32_t)dv.w & 0xffu, nwB = ((uint32_t)dv.w >> 8) & 0xffu;
        const bool wide = uv.z >= 2;
        const uint32_t off = (lane < 8) ? (uint32_t)dv.x + sbeg * (wide ? 128u : 32u * nwA)
                                        : (uint32_t)dv.y + sbeg * (wide ? 64u : 32u * nwB);
        prefetch_l1(reinterpret_cast<const char*>(tab + off) + (lane & 7) * 128);
    }
}

template <bool TILE>
__global__ void __launch_bounds__(PROD_THREADS, 1) k_product_t(const ProdArgs a) {
    extern __shared__ __align__(128) char prod_smem[];
    char* smem = prod_smem;
    char* s1 = smem + SMO_S1;
    char* s2 = smem + SMO_S2;
    Unit3Rec* s_units = reinterpret_cast<Unit3Rec*>(smem + SMO_UNITS);
    Diag3Rec* s_diags = reinterpret_cast<Diag3Rec*>(smem + SMO_DIAGS);
    volatile ProdCtrl* ctl = reinterpret_cast<volatile ProdCtrl*>(smem + SMO_CTRL);
    void* mbar1 = smem + SMO_CTRL + offsetof(ProdCtrl, mbar1);
    void* mbar2 = smem + SMO_CTRL + offsetof(ProdCtrl, mbar2);
    int* next_unit = reinterpret_cast<int*>(smem + SMO_CTRL + offsetof(ProdCtrl, next_unit));
    const int tid = threadIdx.x;
    const size_t scr_stride = (size_t)a.max_pair_units * 256;
    double2* scr0 = a.scratch + (size_t)blockIdx.x * PROD_NBUF * scr_stride;

    if (tid == 0) {
        mbar_init(mbar1, 1);
        mbar_init(mbar2, 1);
        ctl->qtask[0] = (long long)atomicAdd(a.counter, 1ull);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= PROD_CTHREADS) {
        // ---------------- epilogue warps: combine item i while the compute warps run item i+1
        const int et = tid - PROD_CTHREADS;
        for (unsigned it = 0;; ++it) {
            const int b = it % PROD_NBUF;
            named_sync(BAR_FULL0 + b, PROD_THREADS);
            const int ip = ctl->meta_pair[b];
            if (ip < 0) break;
            const size_t q = (size_t)ctl->meta_q[b];
            combine_item<TILE>(a, ip, q, ctl->meta_acc[b] != 0, scr0 + b * scr_stride, et, smem + SMO_EPI);
            named_arrive(BAR_EMPTY0 + b, PROD_THREADS);
        }
        return;
    }

    // ---------------- compute warps
    const int lane = tid & 31;
    uint32_t ph1 = 0, ph2 = 0; // phase parities of the two staging barriers
    int pos = 0;               // position in the chain of sink pairs
    unsigned ntask = 0;
    long long qt = 0;
    size_t q = 0, mq = 0;
    int cbase = 0, clen = 1;
    size_t xs = 0, nsites = (size_t)a.L * a.L * a.L; // direct mode: site X of the shifted sum
    int4 nh0 = make_int4(0, 0, 0, 0), nh1 = nh0, nh2 = nh0; // next chain record
    for (unsigned it = 0;; ++it) {
        const int b = it % PROD_NBUF;
        named_sync(BAR_COMPUTE, PROD_CTHREADS); // the staged blocks and unit records of the previous item are consumed
        if (pos == 0) {
            if (!a.direct || xs == 0) qt = ctl->qtask[ntask & 1]; // new task
            if (qt < a.ntasks) {
                if (TILE) { // one sink pair, every momentum of the list
                    q = (size_t)__ldg(a.qorder + qt);
                    mq = minus_q(a.L, q);
                    cbase = a.chain_base;
                    clen = 1;
                } else if (a.direct) { // task = displacement r = qt; this pass of the chain: site X = xs
                    mq = xs;
                    q = shifted_site(a.L, xs, (size_t)qt);
                    cbase = 0;
                    clen = a.chain_full_n;
                } else {
                    q = (size_t)__ldg(a.qorder + qt);
                    mq = minus_q(a.L, q);
                    // momenta q > -q leave the pairs of identical sink baryons to the task of -q
                    cbase = (mq < q) ? a.chain_full_n : 0;
                    clen = (mq < q) ? a.chain_half_n : a.chain_full_n;
                }
            }
        }
        if (it >= PROD_NBUF) named_sync(BAR_EMPTY0 + b, PROD_THREADS); // scratch buffer b and its descriptor are free again
        if (qt >= a.ntasks) { // no work left: tell the epilogue warps and leave
            if (tid == 0) ctl->meta_pair[b] = -1;
            __threadfence_block();
            named_arrive(BAR_FULL0 + b, PROD_THREADS);
            break;
        }
        // chain record of this item (prefetched during the previous item of the same momentum task)
        const int4* crec = reinterpret_cast<const int4*>(a.chain + cbase + pos);
        const int4 h0 = (pos > 0) ? nh0 : __ldg(crec);
        const int ip = h0.x, load1 = h0.y, load2 = h0.z, nunits = h0.w;
        const int4 h1 = (pos > 0) ? nh1 : __ldg(crec + 1); // unit_begin, ndiags, diag_begin
        if (tid == 0) {
            const int4 h2 = (pos > 0) ? nh2 : __ldg(crec + 2); // buf1, off1, buf2, off2
            *next_unit = 0;
            ctl->meta_q[b] = a.direct ? (int)qt : (int)q; // row of Ft this item goes to
            ctl->meta_pair[b] = ip;
            ctl->meta_acc[b] = (a.direct && xs > 0) ? 1 : 0;
            // unit and diagram records of the pair ride on the first staging barrier of the item
            const uint32_t ubytes = (uint32_t)nunits * (uint32_t)sizeof(Unit3Rec);
            const uint32_t dbytes = (uint32_t)h1.y * (uint32_t)sizeof(Diag3Rec);
            void* rbar = load1 ? mbar1 : mbar2;
            constexpr int NPL = TILE ? 2 : 4; // staged sink-spin planes per side
            if (load1) mbar_expect_tx(mbar1, NPL * PLANE_BYTES + ubytes + dbytes);
            if (load2) mbar_expect_tx(mbar2, NPL * PLANE_BYTES + (load1 ? 0u : ubytes + dbytes));
            if (load1) {
                const char* g1 = TILE ? reinterpret_cast<const char*>(a.c1 + q * (size_t)(2 * SM_PLANE))
                                      : reinterpret_cast<const char*>((h2.x ? a.Be + q * a.Re : a.Bc + q * a.Rc) + h2.y);
#pragma unroll
                for (int p = 0; p < NPL; ++p) bulk_g2s(s1 + p * PLANE_BYTES, g1 + p * PLANE_BYTES, PLANE_BYTES, mbar1);
            }
            if (load2) {
                const char* g2 = TILE ? reinterpret_cast<const char*>(a.c2 + mq * (size_t)(2 * SM_PLANE))
                                      : reinterpret_cast<const char*>((h2.z ? a.Be + mq * a.Re : a.Bc + mq * a.Rc) + h2.w);
#pragma unroll
                for (int p = 0; p < NPL; ++p) bulk_g2s(s2 + p * PLANE_BYTES, g2 + p * PLANE_BYTES, PLANE_BYTES, mbar2);
            }
            bulk_g2s(s_units, a.units + h1.x, ubytes, rbar);
            bulk_g2s(s_diags, a.diags + h1.z, dbytes, rbar);
            if (pos == 0 && (!a.direct || xs == 0)) ctl->qtask[(ntask + 1) & 1] = (long long)atomicAdd(a.counter, 1ull); // next task
            if (pos + 1 < clen) nh2 = __ldg(crec + 5);
            // the blocks the NEXT item will stage are pulled into L2 now, one item ahead of their bulk copy (69.8 -> 69.3 ms)
            if (!TILE && !a.direct) {
                if (pos + 1 < clen) {
                    const int4 n0 = __ldg(crec + 3);
                    if (n0.y) bulk_prefetch_l2((nh2.x ? a.Be + q * a.Re : a.Bc + q * a.Rc) + nh2.y, BLOCK_BYTES);
                    if (n0.z) bulk_prefetch_l2((nh2.z ? a.Be + mq * a.Re : a.Bc + mq * a.Rc) + nh2.w, BLOCK_BYTES);
                } else {
                    const long long nqt = ctl->qtask[(ntask + 1) & 1];
                    if (nqt < a.ntasks) {
                        const size_t q2 = (size_t)__ldg(a.qorder + nqt), mq2 = minus_q(a.L, q2);
                        const int4 f2 = __ldg(reinterpret_cast<const int4*>(a.chain + ((mq2 < q2) ? a.chain_full_n : 0)) + 2);
                        bulk_prefetch_l2((f2.x ? a.Be + q2 * a.Re : a.Bc + q2 * a.Rc) + f2.y, BLOCK_BYTES);
                        bulk_prefetch_l2((f2.z ? a.Be + mq2 * a.Re : a.Bc + mq2 * a.Rc) + f2.w, BLOCK_BYTES);
                    }
                }
            }
        }
        if (pos + 1 < clen) { nh0 = __ldg(crec + 3); nh1 = __ldg(crec + 4); }
        // while the copies fly: table heads of the unit this warp will probably start with
        if ((tid >> 5) < nunits) prefetch_unit(a.units + h1.x + (tid >> 5), a.diags + h1.z, a.tab, lane);
        if (load1) { mbar_wait(mbar1, ph1); ph1 ^= 1u; }
        if (load2) { mbar_wait(mbar2, ph2); ph2 ^= 1u; }
        double2* scr = scr0 + b * scr_stride;
        // Table words are the first link of every gather chain and come from L2: the head of the
        // tables of the unit this warp will probably take next (i + number of compute warps) is pulled
        // into L1 while unit i runs -- a hint only, units are still taken from the counter when needed.
        auto grab = [&]() {
            int i = 0;
            if (lane == 0) i = atomicAdd(next_unit, 1);
            return __shfl_sync(0xffffffffu, i, 0);
        };
        int i = grab();
        while (i < nunits) {
            const int4 uv = *reinterpret_cast<const int4*>(s_units + i);
            Unit3Rec u;
            u.diag_begin = uv.x; u.diag_end = uv.y; u.cls = uv.z; u.slot = uv.w;
            if (i + PROD_CWARPS < nunits) prefetch_unit(s_units + i + PROD_CWARPS, s_diags, a.tab, lane);
            double2* out = scr + (size_t)u.slot * 256;
            if (u.cls < 2) run_unit_square<TILE>(u, s_diags, a.tab, s1, s2, out, lane, a.tile_i, a.tile_j);
            else run_unit_wide<TILE>(u, s_diags, a.tab, s1, s2, out, lane, a.tile_i, a.tile_j);
            i = grab();
        }
        __threadfence_block();
        named_arrive(BAR_FULL0 + b, PROD_THREADS); // unit results of this item are in scratch buffer b
        if (++pos == clen) {
            pos = 0;
            if (a.direct && ++xs < nsites) continue; // same displacement, next site X
            xs = 0;
            ++ntask;
        }
    }
}

} // namespace nbs
