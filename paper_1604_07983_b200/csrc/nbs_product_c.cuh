// Pipelined variant of the product kernel (eqs. 4.2-4.3) for the resident plan.
//
// Same arithmetic as k_product_t<false> (nbs_product.cuh): per diagram a complex GEMM over the shared index on
// DMMA.8x8x4, effective-block entries gathered straight into MMA fragments.  What changes is how the blocks
// reach shared memory and how the warps move from one sink pair to the next:
//   * antisymmetric blocks (p, n, Sigma+-, Xi0-) are staged in their COMPACT form (55.5 KB instead of 111 KB),
//     exactly as the block kernel and the forward FFT leave them in HBM: no expansion pass, no second buffer.
//     The gather tables address the compact layout; a mirrored entry changes sides of its (+, -) pair, and the
//     few entries that end up with two terms of one sign carry a flag (bit 31 of the table word) that flips the
//     sign of the loaded value with one integer instruction.
//   * shared memory holds four block slots (a full block takes two).  The host simulated the walk over a task
//     (momentum pair q, -q: full chain, then half chain) and wrote a static program (nbs_tables.hpp, CItem /
//     CLoad): every item knows where its blocks are, which of them it must wait for, and which bulk copies may be
//     issued the moment it is complete.  The warp that completes an item (last to arrive at its counter) issues
//     those copies; nobody waits at an item boundary unless the block it needs is still on its way.  Warps run up
//     to two items ahead of the slowest one, so the tail of a small sink pair is filled with units of the next.
#pragma once
#include "nbs_product.cuh"
#include "nbs_epilogue_c.cuh"

namespace nbs {

// Warp split: 12 compute warps (three per SM sub-partition) + 4 epilogue warps = four warp groups of 128 threads.  The
// CTA is launched with 65536 / 512 = 128 registers per thread; at its first instruction every compute warp group
// raises its budget to C_REG_COMPUTE and the epilogue warp group lowers its own to C_REG_EPILOGUE (setmaxnreg: 12 x
// 32 x 144 + 4 x 32 x 80 = 65536, the whole register file of the SM), so the unit code keeps the registers it needs
// (no spills) while a third compute warp per sub-partition covers more of the latency of a k-step's dependent chain
// (isolated unit code, nbs_probe_kstep: 288 / 551 cycles per k-step and sub-partition with 12 warps against 304 / 576
// with 10).  Measured (profiles/r2_summary.md): 10 + 2 warps at 152 registers 62.0 ms; 12 + 4 at 128 registers without
// setmaxnreg 65.5 (spills); 12 + 4 with 144 / 80 registers 60.1; with units of whole diagrams (build_plan) 58.8.
// Other budgets: 136 / 104 60.9 - 64.2, 152 / 56 64.5 (the epilogue spills).
// The epilogue reads the unit rows with a pipelined reader (nbs_epilogue_c.cuh), C_EPI_ROWS rows per batch, one spin
// component per thread and pass (C_EPI_NM: two components need more than 80 registers).
constexpr int C_CWARPS = 12, C_EWARPS = 4;
constexpr int C_REG_COMPUTE = 144, C_REG_EPILOGUE = 80;
static_assert(C_CWARPS % 4 == 0 && C_EWARPS == 4, "setmaxnreg works on warp groups of four warps");
static_assert(32 * (C_CWARPS * C_REG_COMPUTE + C_EWARPS * C_REG_EPILOGUE) == 65536, "register budgets must add up to the register file");
constexpr int C_EPI_ROWS = 3, C_EPI_NM = 1;
constexpr int C_CTHREADS = C_CWARPS * 32, C_ETHREADS = C_EWARPS * 32, C_THREADS = C_CTHREADS + C_ETHREADS;

struct CProdArgs {
    ProdArgs base;        // pairs, pair_chans, Ft, ch_begin, nch_out, L, scratch, max_pair_units, counter (epilogue and bookkeeping)
    const double2* B;     // [V][R] momentum-space blocks, compact rows
    size_t R;
    const int* slot_off;  // [slots] complex offset inside the row of the block staged for a slot (isospin limit: the partner's)
    const double* pair_sign; // [pairs] +-1: product of the signs of the two staged blocks (isospin limit), else +1
    long long ntasks;     // momentum pairs
    const int* qhalf;     // [ntasks] the momenta q <= -q
    const CItem* prog;
    int nitems;
    const CLoad* loads;
    const Unit3Rec* units;
    const Diag3Rec* diags; // compact-table diagram records (Plan::diagsc)
    const uint32_t* tab;   // Plan::tabc, packed words
    uint32_t rec_stride, units_bytes; // record buffer: the item (CItem), unit records at C_ITEM_BYTES, diagram records units_bytes further
};

struct CCtrl {
    unsigned long long bar_slot[C_NSLOT]; // a block has landed in slot s
    unsigned long long bar_rec[C_NREC];   // unit and diagram records of an item have landed
    unsigned long long full[PROD_NBUF];   // all compute warps have written their unit results of the item in ring buffer b
    unsigned long long empty[PROD_NBUF];  // the epilogue warps are done with ring buffer b
    int next_unit[8], done_cnt[8];        // per item in flight (sequence number modulo 8)
    long long qtask[4];                   // task indices of this CTA (task number modulo 4)
    int meta_q[PROD_NBUF], meta_pair[PROD_NBUF];
};
constexpr uint32_t SMC_REC = C_BLOCKS_BYTES; // 222 720: the block slots come first
constexpr uint32_t C_ITEM_BYTES = 48;
static_assert(sizeof(CItem) == C_ITEM_BYTES, "CItem is read as three int4");
inline size_t cprod_smem_bytes(uint32_t rec_stride) {
    return (size_t)SMC_REC + (size_t)C_NREC * rec_stride + EPI_PAIR_BYTES + EPI_CG * sizeof(PairChanRec) + 16 + sizeof(CCtrl);
}

__device__ __forceinline__ void mbar_arrive(void* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// value with its sign flipped if bit 31 of w is set
__device__ __forceinline__ double flipd(double v, uint32_t w) {
    return __hiloint2double(__double2hiint(v) ^ (int)(w & 0x80000000u), __double2loint(v));
}
// One packed table word (nbs_tables.hpp) = one (+, -) pair of gather terms.  p0: the lane's sink-spin plane a of the
// staged block; plane a + 2 lies C_PAIR_BYTES further in both kinds of block (an immediate offset of the load).
template <int NP>
__device__ __forceinline__ void ldc(const char* p0, uint32_t w, double2 (&u)[NP], double2 (&v)[NP]) {
    const uint32_t ox = w & 0x7ff0u, oy = (w >> 16) & 0x7ff0u;
    u[0] = *reinterpret_cast<const double2*>(p0 + ox);
    v[0] = *reinterpret_cast<const double2*>(p0 + oy);
    if (NP == 2) {
        u[NP - 1] = *reinterpret_cast<const double2*>(p0 + ox + C_PAIR_BYTES);
        v[NP - 1] = *reinterpret_cast<const double2*>(p0 + oy + C_PAIR_BYTES);
    }
}
template <int NP, bool FIRST>
__device__ __forceinline__ void subc(const double2 (&u)[NP], const double2 (&v)[NP], uint32_t w, double2 (&out)[NP]) {
    const uint32_t fu = w << 16; // flip flag of the + term to bit 31
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const double dx = flipd(u[p].x, fu) - flipd(v[p].x, w), dy = flipd(u[p].y, fu) - flipd(v[p].y, w);
        if (FIRST) out[p] = make_double2(dx, dy);
        else { out[p].x += dx; out[p].y += dy; }
    }
}
__device__ __forceinline__ uint32_t ldw(const uint32_t* p) { return __ldg(p); }

// -DNBS_PROF: cycle counters of the compute warps, summed over the launch (read by nbs_stage_times, printed to stderr).
// The epilogue warps carry none: clock reads around combine_item slowed the launch from 63 to 97 ms.
#ifdef NBS_PROF
enum { PF_TOTAL, PF_UNITS, PF_EMPTY, PF_REC, PF_SLOT, PF_RELEASE, PF_MULTI, PF_N };
__device__ unsigned long long g_cprof[PF_N];
#define PF_T(var) const long long var = clock64()
#define PF_ADD(idx, t0) pf[idx] += clock64() - (t0)
#else
#define PF_T(var)
#define PF_ADD(idx, t0)
#endif

// Per-lane views of the two staged blocks of an item: a0 = B~1 at the lane's plane (r & 1), b0 the same for B~2;
// w1 / w2 = plane (r & 3) of B~1 / B~2 (operand B of the 64 x 4 classes).
struct CSides { const char *a0, *b0, *w1, *w2; };
// item: the staged CItem (shared memory); words 5-8 = off1, off2, ps1, ps2 (ps: bytes of one plane)
__device__ __forceinline__ CSides make_sides(const char* smem, const int* item, int lane) {
    const uint32_t off1 = (uint32_t)item[5], off2 = (uint32_t)item[6], ps1 = (uint32_t)item[7], ps2 = (uint32_t)item[8];
    const uint32_t r = (uint32_t)lane >> 2;
    CSides sd;
    sd.a0 = smem + off1 + (r & 1u) * ps1;
    sd.b0 = smem + off2 + (r & 1u) * ps2;
    sd.w1 = sd.a0 + ((r >> 1) & 1u) * C_PAIR_BYTES;
    sd.w2 = sd.b0 + ((r >> 1) & 1u) * C_PAIR_BYTES;
    return sd;
}

// L1 prefetch of the head of the two gather tables of a diagram record (dp: shared memory)
__device__ __forceinline__ void prefetch_diag_c(const Diag3Rec* dp, bool wide, const uint32_t* __restrict__ tab, int lane) {
    if (lane < 12) {
        const int4 dv = *reinterpret_cast<const int4*>(dp);
        const uint32_t sbeg = (uint32_t)dv.z & 0xffffu, nwA = (uint32_t)dv.w & 0xffu, nwB = ((uint32_t)dv.w >> 8) & 0xffu;
        const uint32_t off = (lane < 8) ? (uint32_t)dv.x + sbeg * (wide ? 64u : 16u * nwA) : (uint32_t)dv.y + sbeg * (wide ? 16u : 16u * nwB);
        prefetch_l1(reinterpret_cast<const char*>(tab + off) + (lane & 7) * 128);
    }
}

__device__ __forceinline__ void wide_loads_A_c(const char* a0, uint4 w, double2 (&ua)[4][2], double2 (&va)[4][2]) {
    ldc<2>(a0, w.x, ua[0], va[0]);
    ldc<2>(a0, w.y, ua[1], va[1]);
    ldc<2>(a0, w.z, ua[2], va[2]);
    ldc<2>(a0, w.w, ua[3], va[3]);
}
__device__ __forceinline__ void wide_subs_A_c(const double2 (&ua)[4][2], const double2 (&va)[4][2], uint4 w, double2 (&A)[4][2]) {
    subc<2, true>(ua[0], va[0], w.x, A[0]);
    subc<2, true>(ua[1], va[1], w.y, A[1]);
    subc<2, true>(ua[2], va[2], w.z, A[2]);
    subc<2, true>(ua[3], va[3], w.w, A[3]);
}
// B entry (8 gather terms = 4 pairs): the lanes hi = 0 and hi = 1 of one (aY, k) need the same entry, so each gathers
// two of the four pairs and the halves are exchanged with a shuffle (lane ^ 16 flips hi)
__device__ __forceinline__ void wide_loads_B_c(const char* sB, uint2 bw, double2 (&ub)[2][1], double2 (&vb)[2][1]) {
    ldc<1>(sB, bw.x, ub[0], vb[0]);
    ldc<1>(sB, bw.y, ub[1], vb[1]);
}
__device__ __forceinline__ void wide_fold_B_c(const double2 (&ub)[2][1], const double2 (&vb)[2][1], uint2 bw, double2 (&Bv)[1]) {
    double2 part[1];
    subc<1, true>(ub[0], vb[0], bw.x, part);
    subc<1, false>(ub[1], vb[1], bw.y, part);
    const double ox = __shfl_xor_sync(0xffffffffu, part[0].x, 16), oy = __shfl_xor_sync(0xffffffffu, part[0].y, 16);
    Bv[0] = make_double2(part[0].x + ox, part[0].y + oy);
}

__device__ __forceinline__ void run_unit_square_c(const Unit3Rec u, const Diag3Rec* diags, const uint32_t* __restrict__ tab,
                                                  const char* smem, const int* item, double2* __restrict__ out, int lane
#ifdef NBS_PROF
                                                  , long long* pf
#endif
                                                  ) {
    const CSides sd = make_sides(smem, item, lane);
    const int r = lane >> 2, kk = lane & 3, c = r >> 1;
    constexpr int NT = 2;
    AccSquare<NT> acc = {};
    for (int d = u.diag_begin; d < u.diag_end; ++d) {
        const Diag3Rec dr = load_diag(diags + d);
        if (d + 1 < u.diag_end) prefetch_diag_c(diags + d + 1, false, tab, lane);
        const int nsteps = dr.send - dr.sbeg;
        if (dr.nwA == 1) {
            // software pipeline: table words four k-steps ahead in registers, shared-memory gathers one ahead, the
            // operands of k-step s + 1 formed (into the other operand buffer) while the MMAs of k-step s run
            const uint32_t* tA = tab + dr.offA + dr.sbeg * 16 + kk * 4 + c;
            const uint32_t* tB = tab + dr.offB + dr.sbeg * 16 + kk * 4 + c;
            const uint32_t wa0 = ldw(tA), wb0 = ldw(tB);
            uint32_t wa1 = ldw(tA + 16), wb1 = ldw(tB + 16), wa2 = ldw(tA + 32), wb2 = ldw(tB + 32);
            uint32_t wa3 = ldw(tA + 48), wb3 = ldw(tB + 48), wa4 = ldw(tA + 64), wb4 = ldw(tB + 64);
            double2 A0[NT], B0[NT], A1[NT], B1[NT], ua[NT], va[NT], ub[NT], vb[NT];
            ldc<NT>(sd.a0, wa0, ua, va);
            ldc<NT>(sd.b0, wb0, ub, vb);
            subc<NT, true>(ua, va, wa0, A0);
            subc<NT, true>(ub, vb, wb0, B0);
            // one k-step: MMAs on (A, B), operands of the next k-step into (An, Bn)
            auto kstep = [&](const double2 (&A)[NT], const double2 (&B)[NT], double2 (&An)[NT], double2 (&Bn)[NT]) {
                tA += 16; tB += 16;
                ldc<NT>(sd.a0, wa1, ua, va); // k-step s + 1 (one step past the end: a valid, unused entry)
                ldc<NT>(sd.b0, wb1, ub, vb);
                const uint32_t na = ldw(tA + 64), nb = ldw(tB + 64); // k-step s + 5
                double sA[NT], sB[NT];
#pragma unroll
                for (int i = 0; i < NT; ++i) { sA[i] = A[i].x + A[i].y; sB[i] = B[i].x + B[i].y; }
#pragma unroll
                for (int i = 0; i < NT; ++i)
#pragma unroll
                    for (int j = 0; j < NT; ++j) {
                        dmma884(acc.p1[i][j][0], acc.p1[i][j][1], A[i].x, B[j].x);
                        dmma884(acc.p2[i][j][0], acc.p2[i][j][1], A[i].y, B[j].y);
                    }
                subc<NT, true>(ua, va, wa1, An);
                subc<NT, true>(ub, vb, wb1, Bn);
#pragma unroll
                for (int i = 0; i < NT; ++i)
#pragma unroll
                    for (int j = 0; j < NT; ++j) dmma884(acc.p3[i][j][0], acc.p3[i][j][1], sA[i], sB[j]);
                wa1 = wa2; wa2 = wa3; wa3 = wa4; wa4 = na;
                wb1 = wb2; wb2 = wb3; wb3 = wb4; wb4 = nb;
            };
            int s = 0;
            for (; s + 1 < nsteps; s += 2) {
                kstep(A0, B0, A1, B1);
                kstep(A1, B1, A0, B0);
            }
            if (s < nsteps) kstep(A0, B0, A1, B1);
        } else {
            PF_T(t_nw);
            const int nw = dr.nwA; // == nwB (4 or 12 term pairs per entry): 16-byte groups of four words
            const uint4* tA = reinterpret_cast<const uint4*>(tab + dr.offA + ((dr.sbeg * 4 + kk) * 4 + c) * nw);
            const uint4* tB = reinterpret_cast<const uint4*>(tab + dr.offB + ((dr.sbeg * 4 + kk) * 4 + c) * nw);
            for (int s = 0; s < nsteps; ++s, tA += 4 * nw, tB += 4 * nw) {
                double2 A[NT], B[NT], ua[NT], va[NT], ub[NT], vb[NT];
#pragma unroll
                for (int p = 0; p < NT; ++p) A[p] = B[p] = make_double2(0.0, 0.0);
                for (int j = 0; j < nw / 4; ++j) {
                    const uint4 qa = __ldg(tA + j), qb = __ldg(tB + j);
                    const uint32_t xa[4] = {qa.x, qa.y, qa.z, qa.w}, xb[4] = {qb.x, qb.y, qb.z, qb.w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        ldc<NT>(sd.a0, xa[e], ua, va);
                        ldc<NT>(sd.b0, xb[e], ub, vb);
                        subc<NT, false>(ua, va, xa[e], A);
                        subc<NT, false>(ub, vb, xb[e], B);
                    }
                }
                mma_square(acc, A, B);
            }
            PF_ADD(PF_MULTI, t_nw); // time in diagrams with 4 or 12 term pairs per entry (K = 9, 1)
        }
    }
#pragma unroll
    for (int i = 0; i < NT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int a1 = 2 * i + (r & 1), c1 = r >> 1;
                const int cc = 2 * kk + e, a2 = 2 * j + (cc & 1), c2 = cc >> 1;
                const int a3 = u.cls == 0 ? c1 : c2, a4 = u.cls == 0 ? c2 : c1;
                out[((a1 * 4 + a2) * 4 + a3) * 4 + a4] =
                    make_double2(acc.p1[i][j][e] - acc.p2[i][j][e], acc.p3[i][j][e] - acc.p1[i][j][e] - acc.p2[i][j][e]);
            }
}

// 64 x 4 classes, B operand folded one k-step ahead: the fold of step s + 1 (DADDs and a shuffle) is issued at the top of
// step s, from gathers issued during step s - 1, so that the 16 MMAs of a step never wait for it.
__device__ __forceinline__ void run_unit_wide_c(const Unit3Rec u, const Diag3Rec* diags, const uint32_t* __restrict__ tab,
                                                 const char* smem, const int* item, double2* __restrict__ out, int lane) {
    const CSides sd = make_sides(smem, item, lane);
    const int r = lane >> 2, kk = lane & 3, hi = r >> 2;
    const char* a0 = (u.cls == 2) ? sd.a0 : sd.b0; // operand A = the block that carries a3 and a4
    const char* sB = (u.cls == 2) ? sd.w2 : sd.w1; // operand B at the lane's plane aY = r & 3
    constexpr int NJ = 2;
    double acc[NJ * 4][2] = {};
    for (int d = u.diag_begin; d < u.diag_end; ++d) {
        const Diag3Rec dr = load_diag(diags + d); // nwA == 1, nwB == 4
        if (d + 1 < u.diag_end) prefetch_diag_c(diags + d + 1, true, tab, lane);
        const int nsteps = dr.send - dr.sbeg;
        const uint4* tA = reinterpret_cast<const uint4*>(tab + dr.offA) + (dr.sbeg * 4 + kk) * 4 + (r >> 1);
        const uint2* tB = reinterpret_cast<const uint2*>(tab + dr.offB) + (dr.sbeg * 4 + kk) * 2 + hi;
        double2 A[4][NJ], Bc[1], Bn[1], ua[4][NJ], va[4][NJ], ub[2][1], vb[2][1];
        uint4 a_c = __ldg(tA), a_1 = __ldg(tA + 16), a_2 = __ldg(tA + 32);
        uint2 b_c = __ldg(tB), b_1 = __ldg(tB + 8), b_2 = __ldg(tB + 16), b_3 = __ldg(tB + 24);
        wide_loads_A_c(a0, a_c, ua, va);
        wide_loads_B_c(sB, b_c, ub, vb);
        wide_subs_A_c(ua, va, a_c, A);
        wide_fold_B_c(ub, vb, b_c, Bc);   // step 0
        wide_loads_B_c(sB, b_1, ub, vb);  // step 1, folded at the top of step 0
        for (int s = 0; s < nsteps; ++s) {
            tA += 16; tB += 8;
            wide_fold_B_c(ub, vb, b_1, Bn);       // k-step s + 1
            wide_loads_A_c(a0, a_1, ua, va);  // k-step s + 1 (one step past the end: valid, unused entries)
            wide_loads_B_c(sB, b_2, ub, vb);      // k-step s + 2
            const uint4 na = __ldg(tA + 32);      // k-step s + 3
            const uint2 nb = __ldg(tB + 24);      // k-step s + 4
            mma_wide<NJ>(acc, A, Bc[0], hi);
            wide_subs_A_c(ua, va, a_1, A);
            Bc[0] = Bn[0];
            a_c = a_1; a_1 = a_2; a_2 = na;
            b_c = b_1; b_1 = b_2; b_2 = b_3; b_3 = nb;
        }
    }
    double* o = reinterpret_cast<double*>(out);
#pragma unroll
    for (int j = 0; j < NJ; ++j)
#pragma unroll
        for (int g = 0; g < 4; ++g)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int aX = 2 * j + (r & 1), cX = 4 * g + (r >> 1);
                const int cc = 2 * kk + e, part = cc >> 2, ay = cc & 3;
                const int a1s = u.cls == 2 ? aX : ay, a2s = u.cls == 2 ? ay : aX;
                o[2 * ((a1s * 4 + a2s) * 16 + cX) + part] = acc[j * 4 + g][e];
            }
}

// L1 prefetch of the table heads of the first diagram of a unit (urec, drecs: shared memory)
__device__ __forceinline__ void prefetch_unit_c(const Unit3Rec* urec, const Diag3Rec* drecs, const uint32_t* __restrict__ tab, int lane) {
    const int4 uv = *reinterpret_cast<const int4*>(urec);
    prefetch_diag_c(drecs + uv.x, uv.z >= 2, tab, lane);
}

// ALIAS: the channel records carry u <-> d images to write (isospin limit with channel relations, nbs_tables.hpp)
template <bool ALIAS>
__global__ void __launch_bounds__(C_THREADS, 1) k_product_c(const CProdArgs a) {
    extern __shared__ __align__(128) char prod_smem[];
    char* smem = prod_smem;
    char* s_rec = smem + SMC_REC;
    char* s_epi = s_rec + C_NREC * a.rec_stride;
    CCtrl* ctlp = reinterpret_cast<CCtrl*>(s_epi + ((EPI_PAIR_BYTES + EPI_CG * (uint32_t)sizeof(PairChanRec) + 15u) & ~15u));
    volatile CCtrl* ctl = ctlp;
    const int tid = threadIdx.x;
    const size_t scr_stride = (size_t)a.base.max_pair_units * 256;
    double2* scr0 = a.base.scratch + (size_t)blockIdx.x * PROD_NBUF * scr_stride;

    // bulk copies of one release-list entry for the task at momentum q (mq = -q)
    auto issue_load = [&](const CLoad ld, size_t q, size_t mq) {
        const size_t mom = ((ld.src >> 8) & 1) ? mq : q;
        const char* src = reinterpret_cast<const char*>(a.B + mom * a.R + __ldg(a.slot_off + (ld.src & 255)));
        void* bar = &ctlp->bar_slot[ld.bar];
        mbar_expect_tx(bar, ld.bytes);
        // four copies in flight, one per sink-spin plane: a full block is contiguous in shared memory, a compact block
        // has its planes 2, 3 C_PAIR_BYTES after its planes 0, 1 (nbs_tables.hpp)
        const uint32_t part = ld.bytes >> 2;
        const bool full = ld.bytes == BLOCK_BYTES;
#pragma unroll
        for (int p = 0; p < 4; ++p)
            bulk_g2s(smem + ld.dst + (full ? p * part : (p >> 1) * C_PAIR_BYTES + (p & 1) * part), src + (size_t)p * part, part, bar);
    };
    auto issue_records = [&](int pos, int rb) {
        const int4 h0 = __ldg(reinterpret_cast<const int4*>(a.prog + pos));     // pair, nunits, unit_begin, ndiags
        const int4 h1 = __ldg(reinterpret_cast<const int4*>(a.prog + pos) + 1); // diag_begin, ...
        const uint32_t ubytes = (uint32_t)h0.y * (uint32_t)sizeof(Unit3Rec), dbytes = (uint32_t)h0.w * (uint32_t)sizeof(Diag3Rec);
        void* bar = &ctlp->bar_rec[rb];
        mbar_expect_tx(bar, C_ITEM_BYTES + ubytes + dbytes);
        bulk_g2s(s_rec + rb * a.rec_stride, a.prog + pos, C_ITEM_BYTES, bar);
        bulk_g2s(s_rec + rb * a.rec_stride + C_ITEM_BYTES, a.units + h0.z, ubytes, bar);
        bulk_g2s(s_rec + rb * a.rec_stride + C_ITEM_BYTES + a.units_bytes, a.diags + h1.x, dbytes, bar);
    };

    if (tid == 0) {
        for (int i = 0; i < C_NSLOT; ++i) mbar_init(&ctlp->bar_slot[i], 1);
        for (int i = 0; i < C_NREC; ++i) mbar_init(&ctlp->bar_rec[i], 1);
        for (int i = 0; i < PROD_NBUF; ++i) { mbar_init(&ctlp->full[i], C_CWARPS); mbar_init(&ctlp->empty[i], 1); }
        for (int i = 0; i < 8; ++i) { ctl->next_unit[i] = 0; ctl->done_cnt[i] = 0; }
        const long long t0 = (long long)atomicAdd(a.base.counter, 1ull);
        ctl->qtask[0] = t0;
        ctl->qtask[1] = (long long)atomicAdd(a.base.counter, 1ull);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        if (t0 < a.ntasks) {
            // prologue: what the previous task would have issued for this one, and the first record buffers
            const size_t q = (size_t)__ldg(a.qhalf + t0), mq = minus_q(a.base.L, q);
            for (int i = 0; i < a.nitems; ++i) {
                const int4 h2 = __ldg(reinterpret_cast<const int4*>(a.prog + i) + 2); // ps2, flags, rel_begin, rel_end
                for (int j = h2.z; j < h2.w; ++j) {
                    const int4 lv = __ldg(reinterpret_cast<const int4*>(a.loads + j));
                    CLoad ld; ld.src = lv.x; ld.dst = (uint32_t)lv.y; ld.bytes = (uint32_t)lv.z; ld.bar = lv.w;
                    if ((ld.src >> 9) & 1) issue_load(ld, q, mq);
                }
            }
            for (int i = 0; i < C_NREC; ++i) issue_records(i, i);
        }
    }
    __syncthreads();

    if (tid >= C_CTHREADS) {
        // ---------------- epilogue warps: combine item i while the compute warps run the following items
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(C_REG_EPILOGUE));
        const int et = tid - C_CTHREADS;
        for (unsigned it = 0;; ++it) {
            const int b = it % PROD_NBUF;
            mbar_wait(&ctlp->full[b], (it / PROD_NBUF) & 1u);
            const int ip = ctl->meta_pair[b];
            if (ip < 0) break;
            const size_t q = (size_t)ctl->meta_q[b];
            combine_item_c<C_ETHREADS, C_EPI_ROWS, C_EPI_NM, ALIAS>(a.base, ip, q, scr0 + b * scr_stride, et, s_epi, __ldg(a.pair_sign + ip));
            if (et == 0) mbar_arrive(&ctlp->empty[b]); // combine_item ends with a barrier of the epilogue threads
        }
        return;
    }

    // ---------------- compute warps
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(C_REG_COMPUTE));
    const int lane = tid & 31;
#ifdef NBS_PROF
    long long pf[PF_N] = {};
    const long long pf_start = clock64();
#endif
    uint32_t par = 0;       // phase parities of the slot barriers (every warp sees every item)
    unsigned seq = 0;       // items started by this warp
    unsigned ntask = 0;
    long long qt = ctl->qtask[0];
    while (qt < a.ntasks) {
        const size_t q = (size_t)__ldg(a.qhalf + qt), mq = minus_q(a.base.L, q);
        const long long qn = ctl->qtask[(ntask + 1) & 3];
        const bool next_valid = qn < a.ntasks;
        for (int pos = 0; pos < a.nitems; ++pos, ++seq) {
            const int b = seq % PROD_NBUF, rb = seq % C_NREC, cs = seq & 7;
            PF_T(t_e);
            if (seq >= PROD_NBUF) mbar_wait(&ctlp->empty[b], ((seq / PROD_NBUF) - 1u) & 1u); // ring buffer b is free again
            PF_ADD(PF_EMPTY, t_e);
            PF_T(t_r);
            mbar_wait(&ctlp->bar_rec[rb], (seq / C_NREC) & 1u);
            PF_ADD(PF_REC, t_r);
            PF_T(t_s);
            // the item, its unit and diagram records: staged in record buffer rb (nothing of it is held in registers
            // across the units)
            const int* item = reinterpret_cast<const int*>(s_rec + rb * a.rec_stride);
            const int nunits = item[1], flags = item[9];
            const int w1 = flags & 7, w2 = (flags >> 3) & 7;
            if (w1) { mbar_wait(&ctlp->bar_slot[w1 - 1], (par >> (w1 - 1)) & 1u); par ^= 1u << (w1 - 1); }
            if (w2) { mbar_wait(&ctlp->bar_slot[w2 - 1], (par >> (w2 - 1)) & 1u); par ^= 1u << (w2 - 1); }
            PF_ADD(PF_SLOT, t_s);
            if (lane == 0) { // every warp writes the same descriptor (the epilogue reads it after the last arrival)
                ctl->meta_q[b] = (int)((flags & 64) ? mq : q);
                ctl->meta_pair[b] = item[0];
            }
            const Unit3Rec* s_units = reinterpret_cast<const Unit3Rec*>(s_rec + rb * a.rec_stride + C_ITEM_BYTES);
            const Diag3Rec* s_diags = reinterpret_cast<const Diag3Rec*>(s_rec + rb * a.rec_stride + C_ITEM_BYTES + a.units_bytes);
            double2* scr = scr0 + b * scr_stride;
            int* next_unit = const_cast<int*>(&ctl->next_unit[cs]);
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
                if (i + C_CWARPS < nunits) prefetch_unit_c(s_units + i + C_CWARPS, s_diags, a.tab, lane);
                double2* out = scr + (size_t)u.slot * 256;
                PF_T(t_u);
#ifdef NBS_PROF
                if (u.cls < 2) run_unit_square_c(u, s_diags, a.tab, smem, item, out, lane, pf);
#else
                if (u.cls < 2) run_unit_square_c(u, s_diags, a.tab, smem, item, out, lane);
#endif
                else run_unit_wide_c(u, s_diags, a.tab, smem, item, out, lane);
                PF_ADD(PF_UNITS, t_u);
                i = grab();
            }
            __syncwarp();
            int old = 0;
            if (lane == 0) {
                __threadfence_block();
                mbar_arrive(&ctlp->full[b]);
                old = atomicAdd(const_cast<int*>(&ctl->done_cnt[cs]), 1);
            }
            old = __shfl_sync(0xffffffffu, old, 0);
            PF_T(t_l);
            if (old == C_CWARPS - 1) {
                // this warp completed the item: its blocks and records are free.  Lanes issue the release list in
                // parallel; lane 31 loads the records of the item C_NREC positions ahead into the buffer just vacated.
                __threadfence_block();
                if (lane == 0) { ctl->done_cnt[cs] = 0; ctl->next_unit[cs] = 0; }
                if (lane == 30 && pos == 0) ctl->qtask[(ntask + 2) & 3] = (long long)atomicAdd(a.base.counter, 1ull);
                __threadfence_block();
                const int rel_begin = item[10], nrel = item[11] - item[10];
                if (lane < nrel) {
                    const int4 lv = __ldg(reinterpret_cast<const int4*>(a.loads + rel_begin + lane));
                    CLoad ld; ld.src = lv.x; ld.dst = (uint32_t)lv.y; ld.bytes = (uint32_t)lv.z; ld.bar = lv.w;
                    if (!((ld.src >> 9) & 1)) issue_load(ld, q, mq);
                    else if (next_valid) {
                        const size_t q2 = (size_t)__ldg(a.qhalf + qn);
                        issue_load(ld, q2, minus_q(a.base.L, q2));
                    }
                }
                // the loads the NEXT item will release are pulled into L2 now, one item ahead of their bulk copies
                // (a load that has to wait for the item before it -- no free slot -- then costs an L2 round trip only)
                if (lane >= 16 && lane < 24 && pos + 1 < a.nitems) {
                    const int4 nh2 = __ldg(reinterpret_cast<const int4*>(a.prog + pos + 1) + 2); // ps2, flags, rel_begin, rel_end
                    const int j = nh2.z + (lane - 16);
                    if (j < nh2.w) {
                        const int4 lv = __ldg(reinterpret_cast<const int4*>(a.loads + j));
                        const bool nxt = (lv.x >> 9) & 1;
                        if (!nxt || next_valid) {
                            const size_t qq = nxt ? (size_t)__ldg(a.qhalf + qn) : q;
                            const size_t mom = ((lv.x >> 8) & 1) ? minus_q(a.base.L, qq) : qq;
                            bulk_prefetch_l2(a.B + mom * a.R + __ldg(a.slot_off + (lv.x & 255)), (uint32_t)lv.z);
                        }
                    }
                }
                if (lane == 31) {
                    const int pr = pos + C_NREC;
                    if (pr < a.nitems) issue_records(pr, rb);
                    else if (next_valid) issue_records(pr - a.nitems, rb);
                }
                __threadfence_block();
            }
            __syncwarp();
            PF_ADD(PF_RELEASE, t_l);
        }
        ++ntask;
        qt = qn;
    }
#ifdef NBS_PROF
    pf[PF_TOTAL] = clock64() - pf_start;
    if (lane == 0)
        for (int i = 0; i < PF_N; ++i) atomicAdd(&g_cprof[i], (unsigned long long)pf[i]);
#endif
    // no work left: tell the epilogue warps (every warp arrives; lane 0 of each writes the same end marker)
    {
        const int b = seq % PROD_NBUF;
        if (seq >= PROD_NBUF) mbar_wait(&ctlp->empty[b], ((seq / PROD_NBUF) - 1u) & 1u);
        if (lane == 0) {
            ctl->meta_pair[b] = -1;
            __threadfence_block();
            mbar_arrive(&ctlp->full[b]);
        }
    }
}

} // namespace nbs
