// (ii)+(iii) EffectiveBaryonBlocks fused into MultiplicationEffectiveBlocks, eqs. 4.2-4.3
// (PAPER.md:104-115), on the FP64 tensor pipe (DMMA.8x8x4, the native FP64 MMA of sm_100a).
//
// Per diagram d the sum over the shared index xi~_d is a small complex GEMM (eq. 4.3)
//     out[m][n] += sum_k  eff1[m][k] * eff2[n][k],   m = (a1, carried spins), n = (a2, carried spins)
// of shape 16 x 16 x K or 64 x 4 x K (K = 1, 9, 36, 144).  One warp owns a whole
// diagram: every effective-block entry (a signed sum of 2, 8 or 24 normal-block entries, eq. 4.2)
// is gathered from shared memory exactly once, straight into the lane that holds it as an MMA
// fragment, and is then used by 8 output columns through the tensor pipe.  The effective blocks
// never exist in memory.
//
// Persistent kernel, one CTA per SM.  A CTA takes work items (momentum q, sink pair) from a global
// counter; items are ordered so that q and -q are adjacent (B~1(q), B~2(-q) and B~1(-q), B~2(q) of
// the 14 sink pairs then hit L2).  For an item the CTA stages B~1(q) and B~2(-q) (2 x 110 KB) in
// shared memory; its warps take "units" (a few diagrams of one elementary correlator with one
// accumulator layout) from a shared-memory counter, accumulate them in registers and write each
// unit's 256 spin components to an L2-resident scratch; finally the CTA sums units per elementary
// correlator and writes the channel correlators (eqs. 2.2-2.3 coefficients) in a fixed order, so
// the result is bitwise reproducible.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "nbs_tables.hpp"

namespace nbs {

constexpr int PROD2_WARPS = 8;
constexpr int PROD2_THREADS = PROD2_WARPS * 32;
constexpr size_t PROD2_SMEM = 2 * (size_t)SM_BLOCK * sizeof(double2) + 256;

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__device__ __forceinline__ double flip(double v, unsigned s) { // s = 0 or 0x80000000: v or -v
    return __hiloint2double(__double2hiint(v) ^ (int)s, __double2loint(v));
}
__device__ __forceinline__ double2 flip2(double2 v, unsigned s) { return make_double2(flip(v.x, s), flip(v.y, s)); }

// One table word = two gather terms (bit 15 / 31: minus sign; low 11 bits: sm_index of the triple).
// raw_load issues the shared-memory loads for NP sink-spin planes, raw_add folds them (signed) into
// out: splitting the two lets the loads of the next k-step fly under the MMAs of the current one.
template <int NP>
__device__ __forceinline__ void raw_load(const double2* __restrict__ base, int stride, uint32_t w,
                                         double2 (&u)[NP], double2 (&v)[NP]) {
    const unsigned i0 = w & 0x7ffu, i1 = (w >> 16) & 0x7ffu;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        u[p] = base[p * stride + i0];
        v[p] = base[p * stride + i1];
    }
}
template <int NP, bool FIRST>
__device__ __forceinline__ void raw_add(uint32_t w, const double2 (&u)[NP], const double2 (&v)[NP],
                                        double2 (&out)[NP]) {
    const unsigned s0 = (w & 0x8000u) << 16, s1 = w & 0x80000000u;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const double2 a = flip2(u[p], s0), b = flip2(v[p], s1);
        if (FIRST) out[p] = make_double2(a.x + b.x, a.y + b.y);
        else { out[p].x += a.x + b.x; out[p].y += a.y + b.y; }
    }
}

// Signed gather of one effective-block entry (eq. 4.2) with a run-time number of table words.
template <int NP>
__device__ __forceinline__ void gather(const double2* __restrict__ base, int stride,
                                       const uint32_t* __restrict__ words, int nw, double2 (&out)[NP]) {
    double2 u[NP], v[NP];
    uint32_t w = __ldg(words);
    raw_load<NP>(base, stride, w, u, v);
    raw_add<NP, true>(w, u, v, out);
    for (int j = 1; j < nw; ++j) {
        w = __ldg(words + j);
        raw_load<NP>(base, stride, w, u, v);
        raw_add<NP, false>(w, u, v, out);
    }
}

// ---- classes 0, 1: 16 x 16 outputs -----------------------------------------------------------
// MMA row = 2*c1 + (a1 & 1) in tile i = a1 >> 1 (from B~1), MMA column likewise from B~2; lane =
// 4*row + k.  The 8 lanes of a quarter warp are 2 adjacent planes x 4 consecutive k: no conflicts.
struct AccSquare {
    double re[2][2][2], im[2][2][2];
};
__device__ __forceinline__ void mma_square(AccSquare& c, const double2 (&A)[2], const double2 (&B)[2]) {
    const double nBy[2] = {flip(B[0].y, 0x80000000u), flip(B[1].y, 0x80000000u)};
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            dmma884(c.re[i][j][0], c.re[i][j][1], A[i].x, B[j].x);
            dmma884(c.im[i][j][0], c.im[i][j][1], A[i].x, B[j].y);
        }
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            dmma884(c.re[i][j][0], c.re[i][j][1], A[i].y, nBy[j]);
            dmma884(c.im[i][j][0], c.im[i][j][1], A[i].y, B[j].x);
        }
}

__device__ __forceinline__ void run_unit_square(const Unit2Rec u, const Diag2Rec* __restrict__ diags,
                                                const uint32_t* __restrict__ tab, const double2* s1,
                                                const double2* s2, double2* __restrict__ out, int lane) {
    const int r = lane >> 2, kk = lane & 3, c = r >> 1;
    const double2* pA = s1 + (r & 1) * SM_PLANE;
    const double2* pB = s2 + (r & 1) * SM_PLANE;
    const double2 zero = make_double2(0.0, 0.0);
    AccSquare acc = {};
    for (int d = u.diag_begin; d < u.diag_end; ++d) {
        const Diag2Rec dr = diags[d];
        if (dr.nA == 2 && dr.nB == 2) {
            // software pipeline: table words two k-steps ahead, shared-memory gathers one ahead
            const uint32_t* tA = tab + dr.offA + (dr.kbeg + kk) * 4 + c;
            const uint32_t* tB = tab + dr.offB + (dr.kbeg + kk) * 4 + c;
            uint32_t wa = __ldg(tA), wb = __ldg(tB);
            double2 A[2], B[2], ua[2], va[2], ub[2], vb[2];
            raw_load<2>(pA, 2 * SM_PLANE, wa, ua, va);
            raw_load<2>(pB, 2 * SM_PLANE, wb, ub, vb);
            uint32_t na = __ldg(tA + 16), nb = __ldg(tB + 16);
            raw_add<2, true>(wa, ua, va, A);
            raw_add<2, true>(wb, ub, vb, B);
            if (dr.kbeg + kk >= dr.K) A[0] = A[1] = B[0] = B[1] = zero;
            for (int k0 = dr.kbeg; k0 < dr.kend; k0 += 4) {
                tA += 16; tB += 16;
                wa = na; wb = nb;
                raw_load<2>(pA, 2 * SM_PLANE, wa, ua, va);
                raw_load<2>(pB, 2 * SM_PLANE, wb, ub, vb);
                na = __ldg(tA + 16); nb = __ldg(tB + 16);
                mma_square(acc, A, B);
                raw_add<2, true>(wa, ua, va, A);
                raw_add<2, true>(wb, ub, vb, B);
                if (k0 + 4 + kk >= dr.K) A[0] = A[1] = B[0] = B[1] = zero;
            }
        } else {
            const int nwA = dr.nA >> 1, nwB = dr.nB >> 1;
            const uint32_t* tA = tab + dr.offA + ((dr.kbeg + kk) * 4 + c) * nwA;
            const uint32_t* tB = tab + dr.offB + ((dr.kbeg + kk) * 4 + c) * nwB;
            for (int k0 = dr.kbeg; k0 < dr.kend; k0 += 4, tA += 16 * nwA, tB += 16 * nwB) {
                double2 A[2], B[2];
                gather<2>(pA, 2 * SM_PLANE, tA, nwA, A);
                gather<2>(pB, 2 * SM_PLANE, tB, nwB, B);
                if (k0 + kk >= dr.K) A[0] = A[1] = B[0] = B[1] = zero; // padded k: contributes nothing
                mma_square(acc, A, B);
            }
        }
    }
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int a1 = 2 * i + (r & 1), c1 = r >> 1;
                const int cc = 2 * kk + e, a2 = 2 * j + (cc & 1), c2 = cc >> 1;
                const int a3 = u.cls == 0 ? c1 : c2, a4 = u.cls == 0 ? c2 : c1;
                out[((a1 * 4 + a2) * 4 + a3) * 4 + a4] = make_double2(acc.re[i][j][e], acc.im[i][j][e]);
            }
}

// ---- classes 2, 3: 64 x 4 outputs ------------------------------------------------------------
// Operand A = the effective block that carries a3 and a4: row m = (aX, cX = a3*4 + a4); tile
// (j, g) holds aX in {2j, 2j+1}, cX in {4g .. 4g+3}; MMA row = 2*(cX & 3) + (aX & 1).  Operand B =
// the other effective block (n = aY).  The 8 MMA columns hold [Re | Im] of the 4 outputs:
//   C += Ar [Br | Bi];  C += Ai [-Bi | Br].
__device__ __forceinline__ void mma_wide(double (&acc)[8][2], const double2 (&A)[4][2], double2 Bv, int hi) {
    const double b1 = hi ? Bv.y : Bv.x;
    const double b2 = hi ? Bv.x : flip(Bv.y, 0x80000000u);
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
        for (int j = 0; j < 2; ++j) dmma884(acc[j * 4 + g][0], acc[j * 4 + g][1], A[g][j].x, b1);
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
        for (int j = 0; j < 2; ++j) dmma884(acc[j * 4 + g][0], acc[j * 4 + g][1], A[g][j].y, b2);
}

__device__ __forceinline__ void run_unit_wide(const Unit2Rec u, const Diag2Rec* __restrict__ diags,
                                              const uint32_t* __restrict__ tab, const double2* s1,
                                              const double2* s2, double2* __restrict__ out, int lane) {
    const int r = lane >> 2, kk = lane & 3, aY = r & 3, hi = r >> 2, cg = r >> 1;
    const double2* pA = (u.cls == 2 ? s1 : s2) + (r & 1) * SM_PLANE;
    const double2* pB = (u.cls == 2 ? s2 : s1) + aY * SM_PLANE;
    const double2 zero = make_double2(0.0, 0.0);
    double acc[8][2] = {};
    for (int d = u.diag_begin; d < u.diag_end; ++d) {
        const Diag2Rec dr = diags[d];
        if (dr.nA == 2 && dr.nB == 8) {
            const uint32_t* tA = tab + dr.offA + (dr.kbeg + kk) * 16 + cg;
            const uint4* tB = reinterpret_cast<const uint4*>(tab + dr.offB) + (dr.kbeg + kk);
            uint32_t wa[4];
            uint4 wb = __ldg(tB);
#pragma unroll
            for (int g = 0; g < 4; ++g) wa[g] = __ldg(tA + 4 * g);
            double2 A[4][2], Bv[1], ua[4][2], va[4][2], ub[4][1], vb[4][1];
#pragma unroll
            for (int g = 0; g < 4; ++g) raw_load<2>(pA, 2 * SM_PLANE, wa[g], ua[g], va[g]);
            raw_load<1>(pB, 0, wb.x, ub[0], vb[0]);
            raw_load<1>(pB, 0, wb.y, ub[1], vb[1]);
            raw_load<1>(pB, 0, wb.z, ub[2], vb[2]);
            raw_load<1>(pB, 0, wb.w, ub[3], vb[3]);
            uint32_t na[4];
            uint4 nb = __ldg(tB + 4);
#pragma unroll
            for (int g = 0; g < 4; ++g) na[g] = __ldg(tA + 64 + 4 * g);
#pragma unroll
            for (int g = 0; g < 4; ++g) raw_add<2, true>(wa[g], ua[g], va[g], A[g]);
            raw_add<1, true>(wb.x, ub[0], vb[0], Bv);
            raw_add<1, false>(wb.y, ub[1], vb[1], Bv);
            raw_add<1, false>(wb.z, ub[2], vb[2], Bv);
            raw_add<1, false>(wb.w, ub[3], vb[3], Bv);
            if (dr.kbeg + kk >= dr.K) {
#pragma unroll
                for (int g = 0; g < 4; ++g) A[g][0] = A[g][1] = zero;
                Bv[0] = zero;
            }
            for (int k0 = dr.kbeg; k0 < dr.kend; k0 += 4) {
                tA += 64; tB += 4;
#pragma unroll
                for (int g = 0; g < 4; ++g) wa[g] = na[g];
                wb = nb;
#pragma unroll
                for (int g = 0; g < 4; ++g) raw_load<2>(pA, 2 * SM_PLANE, wa[g], ua[g], va[g]);
                raw_load<1>(pB, 0, wb.x, ub[0], vb[0]);
                raw_load<1>(pB, 0, wb.y, ub[1], vb[1]);
                raw_load<1>(pB, 0, wb.z, ub[2], vb[2]);
                raw_load<1>(pB, 0, wb.w, ub[3], vb[3]);
                nb = __ldg(tB + 4);
#pragma unroll
                for (int g = 0; g < 4; ++g) na[g] = __ldg(tA + 64 + 4 * g);
                mma_wide(acc, A, Bv[0], hi);
#pragma unroll
                for (int g = 0; g < 4; ++g) raw_add<2, true>(wa[g], ua[g], va[g], A[g]);
                raw_add<1, true>(wb.x, ub[0], vb[0], Bv);
                raw_add<1, false>(wb.y, ub[1], vb[1], Bv);
                raw_add<1, false>(wb.z, ub[2], vb[2], Bv);
                raw_add<1, false>(wb.w, ub[3], vb[3], Bv);
                if (k0 + 4 + kk >= dr.K) {
#pragma unroll
                    for (int g = 0; g < 4; ++g) A[g][0] = A[g][1] = zero;
                    Bv[0] = zero;
                }
            }
        } else {
            const int nwA = dr.nA >> 1, nwB = dr.nB >> 1;
            const uint32_t* tA = tab + dr.offA + ((dr.kbeg + kk) * 16 + cg) * nwA;
            const uint32_t* tB = tab + dr.offB + (dr.kbeg + kk) * nwB;
            for (int k0 = dr.kbeg; k0 < dr.kend; k0 += 4, tA += 64 * nwA, tB += 4 * nwB) {
                double2 A[4][2], Bv[1];
#pragma unroll
                for (int g = 0; g < 4; ++g) gather<2>(pA, 2 * SM_PLANE, tA + 4 * g * nwA, nwA, A[g]);
                gather<1>(pB, 0, tB, nwB, Bv);
                if (k0 + kk >= dr.K) {
#pragma unroll
                    for (int g = 0; g < 4; ++g) A[g][0] = A[g][1] = zero;
                    Bv[0] = zero;
                }
                mma_wide(acc, A, Bv[0], hi);
            }
        }
    }
    double* o = reinterpret_cast<double*>(out);
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int g = 0; g < 4; ++g)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int aX = 2 * j + (r & 1), cX = 4 * g + (r >> 1);
                const int cc = 2 * kk + e, part = cc >> 2, ay = cc & 3;
                const int a1 = u.cls == 2 ? aX : ay, a2 = u.cls == 2 ? ay : aX;
                o[2 * ((a1 * 4 + a2) * 16 + cX) + part] = acc[j * 4 + g][e];
            }
}

struct Prod2Args {
    const double2* Bq;   // [V][R] momentum-space normal blocks
    size_t R;
    int L;
    int npairs;
    long long nitems;    // V * npairs
    const int* qorder;   // [V] momenta with q and -q adjacent
    const Pair2Rec* pairs;
    const Unit2Rec* units;
    const Diag2Rec* diags;
    const uint32_t* tab;
    const int* sched;
    const PairChanRec* pair_chans;
    double2* scratch;    // [gridDim.x][max_pair_units][256]
    int max_pair_units;
    double2* Ft;         // [V][nch_out][256]
    int ch_begin, nch_out;
    unsigned long long* counter; // zeroed before the launch
};

__device__ __forceinline__ size_t minus_q2(int L, size_t q) {
    int x = (int)(q % L), y = (int)((q / L) % L), z = (int)(q / ((size_t)L * L));
    x = x ? L - x : 0; y = y ? L - y : 0; z = z ? L - z : 0;
    return x + (size_t)L * (y + (size_t)L * z);
}

// global block element i = a*1728 + (xi1*12 + xi2)*12 + xi3  ->  staged position (sm_index)
__device__ __forceinline__ int staged_index(int i) {
    const int a = i / NTRIPLE, t = i - a * NTRIPLE;
    const int xi1 = t / 144, rem = t - xi1 * 144, xi2 = rem / 12, xi3 = rem - xi2 * 12;
    int x3 = xi3 + xi2;
    x3 = x3 >= 12 ? x3 - 12 : x3;
    return a * SM_PLANE + xi1 * SM_STRIDE1 + xi2 * 12 + x3;
}

__global__ void __launch_bounds__(PROD2_THREADS, 1) k_product_v2(const Prod2Args a) {
    extern __shared__ double2 smem[];
    double2* s1 = smem;
    double2* s2 = smem + SM_BLOCK;
    Pair2Rec* s_pr = reinterpret_cast<Pair2Rec*>(smem + 2 * SM_BLOCK); // 100 bytes
    long long* s_item = reinterpret_cast<long long*>(reinterpret_cast<char*>(s_pr) + 128);
    int* s_next = reinterpret_cast<int*>(s_item + 1);
    const int tid = threadIdx.x, lane = tid & 31;
    double2* scr = a.scratch + (size_t)blockIdx.x * a.max_pair_units * 256;

    for (;;) {
        __syncthreads(); // previous item fully consumed (shared memory, scratch)
        if (tid == 0) {
            *s_item = (long long)atomicAdd(a.counter, 1ull);
            *s_next = 0;
        }
        __syncthreads();
        const long long item = *s_item;
        if (item >= a.nitems) break;
        const size_t q = (size_t)a.qorder[item / a.npairs];
        const int ip = (int)(item % a.npairs);
        if (tid < (int)(sizeof(Pair2Rec) / sizeof(int)))
            reinterpret_cast<int*>(s_pr)[tid] = reinterpret_cast<const int*>(a.pairs + ip)[tid];
        {
            const double2* g1 = a.Bq + q * a.R + (size_t)a.pairs[ip].slot1 * BLOCK_ELEMS;
            const double2* g2 = a.Bq + minus_q2(a.L, q) * a.R + (size_t)a.pairs[ip].slot2 * BLOCK_ELEMS;
#pragma unroll 3
            for (int i = tid; i < BLOCK_ELEMS; i += PROD2_THREADS) { // 6912 = 27 * 256
                const int j = staged_index(i);
                const double2 v1 = __ldcs(g1 + i), v2 = __ldcs(g2 + i);
                s1[j] = v1;
                s2[j] = v2;
            }
        }
        __syncthreads();
        const int nunits = s_pr->nunits;
        const Unit2Rec* units = a.units + s_pr->unit_begin;
        const int* sched = a.sched + s_pr->sched_begin;
        for (;;) {
            int i = 0;
            if (lane == 0) i = atomicAdd(s_next, 1);
            i = __shfl_sync(0xffffffffu, i, 0);
            if (i >= nunits) break;
            const int ul = sched[i];
            const Unit2Rec u = units[ul];
            double2* out = scr + (size_t)ul * 256;
            if (u.cls < 2) run_unit_square(u, a.diags, a.tab, s1, s2, out, lane);
            else run_unit_wide(u, a.diags, a.tab, s1, s2, out, lane);
        }
        __syncthreads(); // all units of this item are in the scratch
        {
            double2 es[MAX_PAIR_ELEMS];
#pragma unroll
            for (int e = 0; e < MAX_PAIR_ELEMS; ++e) {
                es[e] = make_double2(0.0, 0.0);
                if (e < s_pr->nelem)
                    for (int ul = s_pr->elem_unit_begin[e]; ul < s_pr->elem_unit_begin[e + 1]; ++ul) {
                        const double2 v = __ldcg(scr + (size_t)ul * 256 + tid);
                        es[e].x += v.x;
                        es[e].y += v.y;
                    }
            }
            for (int c = 0; c < s_pr->nchan; ++c) {
                const PairChanRec* pc = a.pair_chans + s_pr->chan_begin + c;
                const int ch = pc->ch - a.ch_begin;
                if (ch < 0 || ch >= a.nch_out) continue;
                double2 acc = make_double2(0.0, 0.0);
#pragma unroll
                for (int e = 0; e < MAX_PAIR_ELEMS; ++e) {
                    const double k = pc->coef[e];
                    acc.x = fma(k, es[e].x, acc.x);
                    acc.y = fma(k, es[e].y, acc.y);
                }
                __stcs(a.Ft + (q * a.nch_out + ch) * 256 + tid, acc);
            }
        }
    }
}

} // namespace nbs
