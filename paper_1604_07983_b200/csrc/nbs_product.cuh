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

constexpr int PROD2_WARPS = 16;
constexpr int PROD2_THREADS = PROD2_WARPS * 32;
constexpr size_t PROD2_SMEM = 2 * (size_t)BLOCK_ELEMS * sizeof(double2) + 256;

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__device__ __forceinline__ double flip(double v, unsigned s) { // s = 0 or 0x80000000: v or -v
    return __hiloint2double(__double2hiint(v) ^ (int)s, __double2loint(v));
}

// Signed gather of one effective-block entry (eq. 4.2) for NP sink-spin planes that share the
// table entries: out[p] = sum_t (+-) base[p * stride + triple_t].
template <int NP>
__device__ __forceinline__ void gather(const double2* __restrict__ base, int stride,
                                       const uint32_t* __restrict__ words, int nw, double2 (&out)[NP]) {
    {
        const uint32_t w = __ldg(words);
        const unsigned i0 = w & 0x7ffu, s0 = (w & 0x8000u) << 16;
        const unsigned i1 = (w >> 16) & 0x7ffu, s1 = w & 0x80000000u;
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const double2 u = base[p * stride + i0], v = base[p * stride + i1];
            out[p].x = flip(u.x, s0) + flip(v.x, s1);
            out[p].y = flip(u.y, s0) + flip(v.y, s1);
        }
    }
    for (int j = 1; j < nw; ++j) {
        const uint32_t w = __ldg(words + j);
        const unsigned i0 = w & 0x7ffu, s0 = (w & 0x8000u) << 16;
        const unsigned i1 = (w >> 16) & 0x7ffu, s1 = w & 0x80000000u;
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const double2 u = base[p * stride + i0], v = base[p * stride + i1];
            out[p].x += flip(u.x, s0) + flip(v.x, s1);
            out[p].y += flip(u.y, s0) + flip(v.y, s1);
        }
    }
}

// Classes 0, 1: 16 x 16 outputs.  m = a1*4 + c1 (rows, from B~1), n = a2*4 + c2 (columns, from B~2).
// Tile (i, j) holds a1 in {2i, 2i+1}, a2 in {2j, 2j+1}; lane = 4*row + k.
template <int CLS>
__device__ __forceinline__ void run_unit_square(const Unit2Rec u, const Diag2Rec* __restrict__ diags,
                                                const uint32_t* __restrict__ tab, const double2* s1,
                                                const double2* s2, double2* __restrict__ out, int lane) {
    const int r = lane >> 2, kk = lane & 3, c = r & 3;
    double cre[2][2][2] = {}, cim[2][2][2] = {};
    const double2* pA = s1 + (r >> 2) * NTRIPLE;
    const double2* pB = s2 + (r >> 2) * NTRIPLE;
    for (int d = u.diag_begin; d < u.diag_end; ++d) {
        const Diag2Rec dr = diags[d];
        const int nwA = dr.nA >> 1, nwB = dr.nB >> 1;
        const uint32_t* tA = tab + dr.offA + (kk * 4 + c) * nwA;
        const uint32_t* tB = tab + dr.offB + (kk * 4 + c) * nwB;
        for (int k0 = 0; k0 < dr.Kp; k0 += 4, tA += 16 * nwA, tB += 16 * nwB) {
            double2 A[2], B[2];
            gather<2>(pA, 2 * NTRIPLE, tA, nwA, A);
            gather<2>(pB, 2 * NTRIPLE, tB, nwB, B);
            if (k0 + kk >= dr.K) { // padded k: contributes nothing
                A[0] = A[1] = B[0] = B[1] = make_double2(0.0, 0.0);
            }
            const double nBy[2] = {flip(B[0].y, 0x80000000u), flip(B[1].y, 0x80000000u)};
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    dmma884(cre[i][j][0], cre[i][j][1], A[i].x, B[j].x);
                    dmma884(cim[i][j][0], cim[i][j][1], A[i].x, B[j].y);
                }
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    dmma884(cre[i][j][0], cre[i][j][1], A[i].y, nBy[j]);
                    dmma884(cim[i][j][0], cim[i][j][1], A[i].y, B[j].x);
                }
        }
    }
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int a1 = 2 * i + (r >> 2), c1 = r & 3;
                const int cc = 2 * kk + e, a2 = 2 * j + (cc >> 2), c2 = cc & 3;
                const int a3 = CLS == 0 ? c1 : c2, a4 = CLS == 0 ? c2 : c1;
                out[((a1 * 4 + a2) * 4 + a3) * 4 + a4] = make_double2(cre[i][j][e], cim[i][j][e]);
            }
}

// Classes 2, 3: 64 x 4 outputs.  Operand A = the effective block that carries a3 and a4
// (m = aX*16 + a3*4 + a4, 8 row tiles), operand B = the other one (n = aY).  The 8 MMA columns
// hold [Re | Im] of the 4 outputs: C += Ar [Br | Bi];  C += Ai [-Bi | Br].
template <int CLS>
__device__ __forceinline__ void run_unit_wide(const Unit2Rec u, const Diag2Rec* __restrict__ diags,
                                              const uint32_t* __restrict__ tab, const double2* s1,
                                              const double2* s2, double2* __restrict__ out, int lane) {
    const int r = lane >> 2, kk = lane & 3, aY = r & 3, hi = r >> 2;
    const double2* sA = CLS == 2 ? s1 : s2;
    const double2* sB = (CLS == 2 ? s2 : s1) + aY * NTRIPLE;
    double acc[8][2] = {};
    for (int d = u.diag_begin; d < u.diag_end; ++d) {
        const Diag2Rec dr = diags[d];
        const int nwA = dr.nA >> 1, nwB = dr.nB >> 1;
        const uint32_t* tA = tab + dr.offA + (kk * 16 + r) * nwA;
        const uint32_t* tB = tab + dr.offB + kk * nwB;
        for (int k0 = 0; k0 < dr.Kp; k0 += 4, tA += 64 * nwA, tB += 4 * nwB) {
            double2 A0[4], A1[4], Bv[1];
            gather<4>(sA, NTRIPLE, tA, nwA, A0);
            gather<4>(sA, NTRIPLE, tA + 8 * nwA, nwA, A1);
            gather<1>(sB, 0, tB, nwB, Bv);
            if (k0 + kk >= dr.K) {
#pragma unroll
                for (int p = 0; p < 4; ++p) A0[p] = A1[p] = make_double2(0.0, 0.0);
                Bv[0] = make_double2(0.0, 0.0);
            }
            const double b1 = hi ? Bv[0].y : Bv[0].x;
            const double b2 = hi ? Bv[0].x : flip(Bv[0].y, 0x80000000u);
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                dmma884(acc[2 * p][0], acc[2 * p][1], A0[p].x, b1);
                dmma884(acc[2 * p + 1][0], acc[2 * p + 1][1], A1[p].x, b1);
            }
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                dmma884(acc[2 * p][0], acc[2 * p][1], A0[p].y, b2);
                dmma884(acc[2 * p + 1][0], acc[2 * p + 1][1], A1[p].y, b2);
            }
        }
    }
    double* o = reinterpret_cast<double*>(out);
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int cX = 8 * h + r, cc = 2 * kk + e, part = cc >> 2, ay = cc & 3;
                const int a1 = CLS == 2 ? p : ay, a2 = CLS == 2 ? ay : p;
                o[2 * (((a1 * 4 + a2) * 16) + cX) + part] = acc[2 * p + h][e];
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

__global__ void __launch_bounds__(PROD2_THREADS, 1) k_product_v2(const Prod2Args a) {
    extern __shared__ double2 smem[];
    double2* s1 = smem;
    double2* s2 = smem + BLOCK_ELEMS;
    Pair2Rec* s_pr = reinterpret_cast<Pair2Rec*>(smem + 2 * BLOCK_ELEMS); // 112 bytes
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
        if (tid < (int)(sizeof(Pair2Rec) / sizeof(int))) reinterpret_cast<int*>(s_pr)[tid] = reinterpret_cast<const int*>(a.pairs + ip)[tid];
        {
            const double2* g1 = a.Bq + q * a.R + (size_t)a.pairs[ip].slot1 * BLOCK_ELEMS;
            const double2* g2 = a.Bq + minus_q2(a.L, q) * a.R + (size_t)a.pairs[ip].slot2 * BLOCK_ELEMS;
#pragma unroll 4
            for (int i = tid; i < BLOCK_ELEMS; i += PROD2_THREADS) {
                s1[i] = __ldcs(g1 + i);
                s2[i] = __ldcs(g2 + i);
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
            switch (u.cls) {
            case 0: run_unit_square<0>(u, a.diags, a.tab, s1, s2, out, lane); break;
            case 1: run_unit_square<1>(u, a.diags, a.tab, s1, s2, out, lane); break;
            case 2: run_unit_wide<2>(u, a.diags, a.tab, s1, s2, out, lane); break;
            default: run_unit_wide<3>(u, a.diags, a.tab, s1, s2, out, lane); break;
            }
        }
        __syncthreads(); // all units of this item are in the scratch
        if (tid < 256) {
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
                a.Ft[(q * a.nch_out + ch) * 256 + tid] = acc;
            }
        }
    }
}

} // namespace nbs
