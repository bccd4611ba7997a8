// sm_100a CUDA kernels of the hot path (rows a1-a5 of DESIGN.md).  Complex128 throughout.
//
// Data layout in HBM ("site-major"): every stage keeps all components of one lattice site (or
// momentum q) contiguous:
//   blocks  B[site][slot][staged block]         (row length R = nslots * 6960 complex; a staged block
//                                               = 4 sink-spin planes in the padded, skewed layout
//                                               of nbs_tables.hpp that the product kernel gathers from)
//   Ft      [q][ch][256]                         channel correlators in momentum space
// so that (a) the block kernel writes one site's 110 KB per baryon fully coalesced, (b) the FFT
// runs one 1-D transform per thread with lanes on consecutive components (coalesced, no shared
// memory), and (c) the product kernel stages B~1(q), B~2(-q) with contiguous bulk reads.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>
#include <utility>

#include "nbs_tables.hpp"

namespace nbs {

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ void cfma(double2& acc, double2 a, double2 b) {
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}

// ---------------------------------------------------------------------------------------------
// (i) NormalBaryonBlocks, eq. 4.1.  One CTA per lattice site.
//   phase 1: diquarks D^{f0f1}_c(i,j) = sum_{ab, beta gamma} eps_abc (C g5)_{beta gamma}
//            S_f0[(a,beta), i] S_f1[(b,gamma), j]            -> shared memory (needed types only)
//   phase 2: block[a][xi0 xi1 xi2] = sum_terms coef sum_c D_c(xi_p0, xi_p1) S_f2[(c,a), xi_p2],
//            one half row (2 sink spins of one baryon) at a time: every thread owns a register
//            tile of 2 (spins) x 2 x 2 x 2 (xi0, xi1, xi2) outputs, so each shared-memory operand
//            is used 4 times (0.5 loads per complex MAC for any permutation p); the half row is
//            assembled in shared memory in the staged layout of nbs_tables.hpp (plane a at
//            a*SM_PLANE, triple at sm_index, pads = 0) and copied to HBM fully coalesced.
// ---------------------------------------------------------------------------------------------
struct BTermRec {
    double coef;
    int dq, f2;
    int p0, p1, p2, pad;
};
struct BlockRec {
    int term_begin, term_end;
};

constexpr int BLOCKS_THREADS = 256;
constexpr int BLOCKS_TILES = 216;               // 6 x 6 x 6 tiles of 2 x 2 x 2 source triples
constexpr int BLOCKS_HALF = 2 * SM_PLANE;       // complex entries of a half row
static_assert(AS_BLOCK <= BLOCKS_HALF, "a compact antisymmetric block is assembled in the half-row buffer");
// Shared-memory operand layouts of k_blocks, chosen so that the register tiles of a warp (tile origins
// 2 i per index, lanes on consecutive i) read without bank conflicts: a source index xi sits at
// dq_rank(xi) = (xi & 1) * 6 + (xi >> 1) (even and odd values de-interleaved: the lanes' even origins
// become consecutive), and a diquark row is 13 entries long (odd stride for lanes that walk the rows).
constexpr int DQ_ROW = 13, DQ_C = 12 * DQ_ROW, DQ_SIZE = 3 * DQ_C; // per diquark type: [c][rank(xi)][rank(xi')]
__host__ __device__ constexpr int dq_rank(int xi) { return (xi & 1) * 6 + (xi >> 1); }
constexpr int BLOCKS_MAX_SLOTS = 16; // per-slot records kept in shared memory (there are 11 interpolating fields)
// Register tile of thread `tid` for a block of `kind`: origins (x0, x1, x2) of its 2 x 2 x 2 source triples, first sink
// spin a0 of its two (full kind: 2 * pass), whether the thread has a tile at all.  Full blocks: 216 tiles per pass of two
// sink spins; antisymmetric blocks: one pass, 2 x 126 tiles on or above the diagonal of the antisymmetric slot pair.
struct BlocksTile { int x0, x1, x2, a0; bool active; };
__host__ __device__ inline BlocksTile blocks_tile(int kind, int tid, int pass) {
    BlocksTile t;
    if (kind == BK_FULL) {
        t.active = tid < BLOCKS_TILES; t.a0 = 2 * pass;
        t.x0 = 2 * (tid / 36); t.x1 = 2 * ((tid / 6) % 6); t.x2 = 2 * (tid % 6);
    } else {
        const int h = tid / 126, tt = tid - h * 126;
        t.active = tid < 252;
        int ia = 0, rem = tt / 6;
        while (rem >= 6 - ia) { rem -= 6 - ia; ++ia; }
        const int ib = ia + rem, ic = tt % 6;
        t.a0 = 2 * h; t.x2 = 2 * ib;
        if (kind == BK_ASYM13) { t.x0 = 2 * ia; t.x1 = 2 * ic; }
        else { t.x1 = 2 * ia; t.x0 = 2 * ic; }
    }
    return t;
}
// Where the 16 results of a thread's tile go in the half-row buffer (index ((a * 2 + e0) * 2 + e1) * 2 + e2), per block
// kind: the same for every slot of a kind, so the host writes them once ([kind][tid][16] uint16, 24 KB, read through L1 /
// L2 as two 16-byte loads per pass) instead of every thread evaluating the layout functions 16 times per pass -- that
// index arithmetic was as many instructions as the arithmetic of a two-term block.  0xffff: no entry (an antisymmetric
// pair with xi_a >= xi_b, a thread without a tile).
constexpr int BLOCKS_OUT_SKIP = 0xffff;
inline void blocks_out_offsets(uint16_t* tab) { // [3][BLOCKS_THREADS][16]
    for (int kind = 0; kind < 3; ++kind)
        for (int tid = 0; tid < 256; ++tid) {
            const BlocksTile t = blocks_tile(kind, tid, 0);
            for (int i = 0; i < 16; ++i) {
                const int a = i >> 3, e0 = (i >> 2) & 1, e1 = (i >> 1) & 1, e2 = i & 1;
                const int xi0 = t.x0 + e0, xi1 = t.x1 + e1, xi2 = t.x2 + e2;
                int off = BLOCKS_OUT_SKIP;
                if (t.active) {
                    if (kind == BK_FULL) off = a * SM_PLANE + sm_index(xi0, xi1, xi2);
                    else {
                        const int xa = (kind == BK_ASYM13) ? xi0 : xi1, xc = (kind == BK_ASYM13) ? xi1 : xi0;
                        if (xa < xi2) off = (t.a0 + a) * AS_PLANE + as_index(xa, xi2, xc);
                    }
                }
                tab[(kind * 256 + tid) * 16 + i] = (uint16_t)off;
            }
        }
}
inline size_t blocks_smem_bytes(int ndq) { return (size_t)(3 * 144 + ndq * DQ_SIZE + BLOCKS_HALF + BLOCKS_MAX_SLOTS) * sizeof(double2); }

// acc[a][e0][e1][e2] += coef * sum_c D_c(xi_P0, xi_P1) * S[(c, a0 + a), xi_P2] over the thread's tile
template <int P0, int P1, int P2>
__device__ __forceinline__ void blocks_term(double2 (&acc)[2][2][2][2], const double2* __restrict__ Dq,
                                            const double2* __restrict__ S2, double coef, int a0, int x0, int x1, int x2) {
    // tile origins as scalars selected at compile time (an int[3] indexed through the run-time switch below
    // was placed in local memory)
    const int xP0 = P0 == 0 ? x0 : P0 == 1 ? x1 : x2, xP1 = P1 == 0 ? x0 : P1 == 1 ? x1 : x2,
              xP2 = P2 == 0 ? x0 : P2 == 1 ? x1 : x2;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double2 Dv[2][2], Sv[2][2];
#pragma unroll
        for (int ja = 0; ja < 2; ++ja)
#pragma unroll
            for (int jb = 0; jb < 2; ++jb) // x even: dq_rank(x + j) = 6 j + x / 2
                Dv[ja][jb] = Dq[c * DQ_C + (6 * ja + (xP0 >> 1)) * DQ_ROW + 6 * jb + (xP1 >> 1)];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const double2 v = S2[(c + 3 * (a0 + a)) * 12 + 6 * j + (xP2 >> 1)];
                Sv[a][j] = make_double2(coef * v.x, coef * v.y);
            }
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int e0 = 0; e0 < 2; ++e0)
#pragma unroll
                for (int e1 = 0; e1 < 2; ++e1)
#pragma unroll
                    for (int e2 = 0; e2 < 2; ++e2) {
                        const int e[3] = {e0, e1, e2};
                        cfma(acc[a][e0][e1][e2], Dv[e[P0]][e[P1]], Sv[a][e[P2]]);
                    }
    }
}

__global__ void __launch_bounds__(BLOCKS_THREADS, 2)
k_blocks(const double2* __restrict__ Su, const double2* __restrict__ Sd, const double2* __restrict__ Ss,
         const int* __restrict__ baryon_of_slot, int nslots, unsigned dq_mask,
         const BlockRec* __restrict__ brec, const BTermRec* __restrict__ bterm,
         const int2* __restrict__ slot_info, const uint16_t* __restrict__ out_off, double2* __restrict__ out, size_t row_stride, int pp) {
    // pp < 0: whole blocks.  pp = 0, 1 (tile-wise plan, one slot): only the sink-spin planes {2 pp, 2 pp + 1},
    // written as a two-plane chunk row (staged planes for a full-kind block, compact planes for an antisymmetric one)
    extern __shared__ double2 smem[];
    const int ndq = __popc(dq_mask);
    double2* sS = smem;                  // [3][144]
    double2* sD = smem + 3 * 144;        // [ndq][3][144], needed diquark types in increasing dq order
    double2* sO = sD + ndq * DQ_SIZE;    // [2][SM_PLANE] half row being assembled
    int4* sSlot = reinterpret_cast<int4*>(sO + BLOCKS_HALF); // [nslots] {term_begin, term_end, row offset, block kind}
    const size_t site = blockIdx.x;
    const int tid = threadIdx.x;
    if (tid < nslots) {
        const BlockRec br = brec[baryon_of_slot[tid]];
        const int2 info = slot_info[tid];
        sSlot[tid] = make_int4(br.term_begin, br.term_end, info.x, info.y);
    }
    for (int i = tid; i < 144; i += BLOCKS_THREADS) {
        const int j = (i / 12) * 12 + dq_rank(i % 12); // source index de-interleaved
        sS[j] = Su[site * 144 + i];
        sS[144 + j] = Sd[site * 144 + i];
        sS[288 + j] = Ss[site * 144 + i];
    }
    __syncthreads();
    for (int idx = tid; idx < ndq * 432; idx += BLOCKS_THREADS) {
        const int slot_dq = idx / 432;
        int dq = 0; // the slot_dq-th set bit of dq_mask
        for (int seen = 0; dq < 9; ++dq)
            if ((dq_mask >> dq) & 1u) { if (seen == slot_dq) break; ++seen; }
        const int rem = idx - slot_dq * 432;
        const int c = rem / 144, ri = (rem / 12) % 12, rj = rem % 12; // positions (ranks) of xi, xi': lanes read consecutive entries
        const double2* S0 = sS + (dq / 3) * 144;
        const double2* S1 = sS + (dq % 3) * 144;
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        double2 acc = make_double2(0.0, 0.0), neg = make_double2(0.0, 0.0);
        // (C g5)_{01} = +1, (C g5)_{10} = -1, (C g5)_{23} = +1, (C g5)_{32} = -1
#pragma unroll
        for (int pr = 0; pr < 2; ++pr) {
            const int be = 2 * pr, ga = 2 * pr + 1;
            cfma(acc, S0[(a + 3 * be) * 12 + ri], S1[(b + 3 * ga) * 12 + rj]); // +eps +cg5
            cfma(neg, S0[(a + 3 * ga) * 12 + ri], S1[(b + 3 * be) * 12 + rj]); // +eps -cg5
            cfma(neg, S0[(b + 3 * be) * 12 + ri], S1[(a + 3 * ga) * 12 + rj]); // -eps +cg5
            cfma(acc, S0[(b + 3 * ga) * 12 + ri], S1[(a + 3 * be) * 12 + rj]); // -eps -cg5
        }
        sD[slot_dq * DQ_SIZE + c * DQ_C + ri * DQ_ROW + rj] = csub(acc, neg);
    }
    __syncthreads();

    double2* orow = out + site * row_stride;
    for (int slot = 0; slot < nslots; ++slot) {
        const int4 rec = sSlot[slot];
        const BlockRec br = {rec.x, rec.y};
        const int2 info = make_int2(rec.z, rec.w); // (offset inside the site row, block kind)
        const int kind = info.y;
        // full blocks: two passes of 2 sink spins, 216 tiles each; antisymmetric blocks (nbs_tables.hpp):
        // one pass, 2 x 126 tiles on or above the diagonal of the antisymmetric slot pair
        const int npass = (kind == BK_FULL) ? 2 : 1;
        for (int pass = 0; pass < npass; ++pass) {
            if (pp >= 0 && kind == BK_FULL && pass != pp) continue; // uniform over the CTA
            const BlocksTile tl = blocks_tile(kind, tid, pass);
            const int x0 = tl.x0, x1 = tl.x1, x2 = tl.x2, a0 = tl.a0;
            const bool active = tl.active && (kind == BK_FULL || pp < 0 || (a0 >> 1) == pp);
            double2 acc[2][2][2][2];
            if (active) {
#pragma unroll
                for (int i = 0; i < 16; ++i) (&acc[0][0][0][0])[i] = make_double2(0.0, 0.0);
                BTermRec nxt = bterm[br.term_begin];
                for (int it = br.term_begin; it < br.term_end; ++it) {
                    const BTermRec bt = nxt; // the next term record is fetched under this term's arithmetic
                    if (it + 1 < br.term_end) nxt = bterm[it + 1];
                    const double2* Dq = sD + __popc(dq_mask & ((1u << bt.dq) - 1u)) * DQ_SIZE;
                    const double2* S2 = sS + bt.f2 * 144;
                    const int perm = bt.p0 * 3 + bt.p1; // (p0, p1) fixes the permutation
                    switch (perm) {
                    case 1: blocks_term<0, 1, 2>(acc, Dq, S2, bt.coef, a0, x0, x1, x2); break;
                    case 2: blocks_term<0, 2, 1>(acc, Dq, S2, bt.coef, a0, x0, x1, x2); break;
                    case 3: blocks_term<1, 0, 2>(acc, Dq, S2, bt.coef, a0, x0, x1, x2); break;
                    case 5: blocks_term<1, 2, 0>(acc, Dq, S2, bt.coef, a0, x0, x1, x2); break;
                    case 6: blocks_term<2, 0, 1>(acc, Dq, S2, bt.coef, a0, x0, x1, x2); break;
                    default: blocks_term<2, 1, 0>(acc, Dq, S2, bt.coef, a0, x0, x1, x2); break;
                    }
                }
            }
            // where the tile's results go (host table, see blocks_out_offsets): fetched under the barrier wait
            const uint4* otab = reinterpret_cast<const uint4*>(out_off + (kind * BLOCKS_THREADS + tid) * 16);
            const uint4 o0 = __ldg(otab), o1 = __ldg(otab + 1);
            // the bulk store of the previous half row (issued by thread 0) must have read sO before it is rewritten
            if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            __syncthreads();
            if (kind == BK_FULL) {
                if (tid < 24) sO[(tid / 12) * SM_PLANE + (tid % 12) * SM_STRIDE1 + 144] = make_double2(0.0, 0.0);
            } else {
                // unused positions of every row (read as the vanishing diagonal by the product kernel) and plane pads
                for (int i = tid; i < 4 * (12 * AS_ROW_PADS + 4); i += BLOCKS_THREADS) {
                    const int pl = i / (12 * AS_ROW_PADS + 4), j = i % (12 * AS_ROW_PADS + 4);
                    const int c = j / AS_ROW_PADS, pos = j < 12 * AS_ROW_PADS ? c * AS_ROW + (as_pad_pos(j % AS_ROW_PADS) + c) % AS_ROW
                                                                              : 12 * AS_ROW + (j - 12 * AS_ROW_PADS);
                    sO[pl * AS_PLANE + pos] = make_double2(0.0, 0.0);
                }
            }
            if (active) {
                const uint32_t ow[8] = {o0.x, o0.y, o0.z, o0.w, o1.x, o1.y, o1.z, o1.w};
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const uint32_t off = (ow[i >> 1] >> (16 * (i & 1))) & 0xffffu;
                    if (off != (uint32_t)BLOCKS_OUT_SKIP) sO[off] = (&acc[0][0][0][0])[i];
                }
            }
            // the half row leaves through the async proxy (one bulk copy shared -> global), under the next pass
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncthreads();
            if (tid == 0) {
                const int n = (kind == BK_FULL) ? BLOCKS_HALF : (pp < 0 ? AS_BLOCK : 2 * AS_PLANE);
                double2* dst = orow + info.x + ((kind == BK_FULL && pp < 0) ? pass * BLOCKS_HALF : 0);
                const double2* src = sO + ((kind != BK_FULL && pp > 0) ? 2 * AS_PLANE : 0);
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n\tcp.async.bulk.commit_group;"
                             :: "l"(dst), "r"((uint32_t)__cvta_generic_to_shared(src)), "r"((uint32_t)(n * sizeof(double2))) : "memory");
            }
        }
    }
    if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); // sO must outlive the last copy
}

// Expansion of the antisymmetric blocks after the forward FFT: compact rows [site][Rc] -> full staged
// blocks [site][Re] (Plan::gather): mirror entries with the sign flipped, pads and diagonal zero.
// Writes are fully coalesced; every compact element is read twice (through L2).
__global__ void __launch_bounds__(256)
k_expand(const double2* __restrict__ compact, size_t Rc, const int* __restrict__ gather, int Re, double2* __restrict__ full) {
    const double2* src = compact + (size_t)blockIdx.x * Rc;
    double2* dst = full + (size_t)blockIdx.x * Re;
    for (int j = threadIdx.x; j < Re; j += 256) {
        const int g = __ldg(gather + j);
        double2 v = make_double2(0.0, 0.0);
        if (g >= 0) {
            v = src[g & 0x3fffffff];
            if (g & (1 << 30)) { v.x = -v.x; v.y = -v.y; }
        }
        dst[j] = v;
    }
}

// Tile-wise plan: the same expansion for a two-plane chunk, in place inside the chunk row (the compact plane pair
// sits at the start of the row of 2 * SM_PLANE entries; Plan::gather_pp).  One CTA per site.
__global__ void __launch_bounds__(256)
k_expand_chunk(double2* __restrict__ chunk, const int* __restrict__ gather) {
    __shared__ double2 buf[2 * AS_PLANE];
    double2* row = chunk + (size_t)blockIdx.x * (2 * SM_PLANE);
    for (int j = threadIdx.x; j < 2 * AS_PLANE; j += 256) buf[j] = row[j];
    __syncthreads();
    for (int j = threadIdx.x; j < 2 * SM_PLANE; j += 256) {
        const int g = __ldg(gather + j);
        double2 v = make_double2(0.0, 0.0);
        if (g >= 0) {
            v = buf[g & 0x3fffffff];
            if (g & (1 << 30)) { v.x = -v.x; v.y = -v.y; }
        }
        row[j] = v;
    }
}

// Staged block rows [site][block of `kind`] -> [site][alpha][xi1][xi2][xi3] (nbs_blocks_x, tests only):
// mirrored entries of an antisymmetric block are reconstructed with their sign.
__global__ void __launch_bounds__(256)
k_unstage(const double2* __restrict__ in, size_t V, int kind, double2* __restrict__ out) {
    const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (idx >= V * BLOCK_ELEMS) return;
    const size_t site = idx / BLOCK_ELEMS;
    const int rem = (int)(idx - site * BLOCK_ELEMS);
    const int al = rem / NTRIPLE, t = rem - al * NTRIPLE;
    const Located loc = locate(kind, t / 144, (t / 12) % 12, t % 12);
    const double2 v = in[site * block_elems(kind) + al * plane_elems(kind) + loc.idx];
    out[idx] = loc.sign > 0 ? v : make_double2(-v.x, -v.y);
}

// ---------------------------------------------------------------------------------------------
// 1-D FFT along one lattice axis, one transform per thread, lanes on consecutive components
// (rows a2 and a5; eq. 2.6).  Forward: sum_x f(x) exp(-i q x); inverse: exp(+i q x)
// times `scale`.  tw[m] = exp(-2 pi i m / L).
// ---------------------------------------------------------------------------------------------
__host__ __device__ constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n >> 1); }
__host__ __device__ constexpr int bitrev(int i, int bits) {
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((i >> b) & 1) << (bits - 1 - b);
    return r;
}

// cos / sin of 2 pi m / 32, m = 0..15, as compile-time constants (they reach the FP64 pipe through
// the constant bank and cost no registers).  exp(-2 pi i k / len) = (tw32_cos, -tw32_sin)(k * 32 / len)
// for every power-of-two len <= 32.
__host__ __device__ constexpr double tw32_quarter(int m) { // cos(2 pi m / 32), 0 <= m <= 8
    constexpr double C[9] = {1.0, 9.807852804032304491e-01, 9.238795325112867561e-01, 8.314696123025452371e-01,
                             7.071067811865475244e-01, 5.555702330196022248e-01, 3.826834323650897717e-01,
                             1.950903220161282679e-01, 0.0};
    return C[m];
}
__host__ __device__ constexpr double tw32_cos(int m) { return m <= 8 ? tw32_quarter(m) : -tw32_quarter(16 - m); }
__host__ __device__ constexpr double tw32_sin(int m) { return m <= 8 ? tw32_quarter(8 - m) : tw32_quarter(m - 8); }

// Compile-time loop: every array index below is a constant, so the L points stay in registers
// (a run-time-indexed double2[32] would be placed in local memory).
template <int... Is, class F>
__device__ __forceinline__ void static_for(std::integer_sequence<int, Is...>, F&& f) {
    (f(std::integral_constant<int, Is>{}), ...);
}

template <int L, bool INV>
__device__ __forceinline__ void fft_inreg(double2 (&a)[L], const double2* __restrict__ tw) {
    constexpr int LOG = ilog2(L);
    static_for(std::make_integer_sequence<int, L>{}, [&](auto ic) {
        constexpr int i = decltype(ic)::value, j = bitrev(i, LOG);
        if constexpr (i < j) { const double2 tmp = a[i]; a[i] = a[j]; a[j] = tmp; }
    });
    static_for(std::make_integer_sequence<int, LOG>{}, [&](auto sc) {
        constexpr int len = 2 << decltype(sc)::value, half = len / 2;
        static_for(std::make_integer_sequence<int, L / 2>{}, [&](auto bc) {
            constexpr int b = decltype(bc)::value, k = b % half, i = (b / half) * len + k;
            const double2 u = a[i];
            double2 v = a[i + half];
            if constexpr (k != 0) {
                if constexpr (4 * k == len) { // w = -i (forward) or +i (inverse)
                    v = INV ? make_double2(-v.y, v.x) : make_double2(v.y, -v.x);
                } else {
                    constexpr double wr = tw32_cos(k * (32 / len)), wi = -tw32_sin(k * (32 / len));
                    v = cmul(v, make_double2(wr, INV ? -wi : wi));
                }
            }
            a[i] = cadd(u, v);
            a[i + half] = csub(u, v);
        });
    });
}

__device__ __forceinline__ void line_geometry(int L, int axis, int line, size_t& s0, size_t& st) {
    int u = line % L, v = line / L;
    if (axis == 0) { s0 = (size_t)L * (u + (size_t)L * v); st = 1; }
    else if (axis == 1) { s0 = u + (size_t)L * L * v; st = L; }
    else { s0 = u + (size_t)L * v; st = (size_t)L * L; }
}

constexpr int FFT_THREADS = 128;

template <int L, bool INV>
__global__ void __launch_bounds__(FFT_THREADS)
k_fft_axis_pow2(double2* __restrict__ data, size_t R, size_t Rn, int axis, const double2* __restrict__ tw, double scale) {
    size_t r = (size_t)blockIdx.x * FFT_THREADS + threadIdx.x; // the first Rn components of rows of length R
    if (r >= Rn) return;
    size_t s0, st;
    line_geometry(L, axis, blockIdx.y, s0, st);
    double2 a[L];
#pragma unroll
    for (int j = 0; j < L; ++j) a[j] = data[(s0 + j * st) * R + r];
    fft_inreg<L, INV>(a, tw);
#pragma unroll
    for (int j = 0; j < L; ++j) {
        double2 v = a[j];
        if (INV) { v.x *= scale; v.y *= scale; }
        data[(s0 + j * st) * R + r] = v;
    }
}

// ---------------------------------------------------------------------------------------------
// L = 3 * L2 with L2 a power of two <= 32 (6, 12, 24, 48 and the 96 of BASELINE.json configs[4]): decimation in
// time by 3.  Three threads share one line: thread s transforms the L2 points x[3 n + s] in registers (the same
// in-register radix-2 code), multiplies by the twiddles w_L^{s k}, and the three partial spectra meet in shared
// memory for the radix-3 butterfly  X[k + L2 m] = sum_s w_3^{s m} (w_L^{s k} Y_s[k]); thread m writes its third
// of the spectrum.  Lanes on consecutive components as in the power-of-two kernel: every access is coalesced.
// tw[m] = exp(-2 pi i m / L), computed in long double on the host.
// ---------------------------------------------------------------------------------------------
constexpr int FFT_R3_COMPS = 64;
template <int L2>
constexpr size_t fft_r3_smem_bytes() { return (size_t)3 * L2 * FFT_R3_COMPS * sizeof(double2); }

template <int L2, bool INV>
__global__ void __launch_bounds__(3 * FFT_R3_COMPS, 2)
k_fft_axis_r3(double2* __restrict__ data, size_t R, size_t Rn, int axis, const double2* __restrict__ tw, double scale) {
    constexpr int L = 3 * L2;
    extern __shared__ double2 smem[]; // [s][k][component]
    const int c = threadIdx.x, s = threadIdx.y;
    const size_t r = (size_t)blockIdx.x * FFT_R3_COMPS + c;
    const bool live = r < Rn;
    size_t s0, st;
    line_geometry(L, axis, blockIdx.y, s0, st);
    double2 a[L2];
    if (live) {
#pragma unroll
        for (int n = 0; n < L2; ++n) a[n] = data[(s0 + (size_t)(3 * n + s) * st) * R + r];
        fft_inreg<L2, INV>(a, nullptr);
#pragma unroll
        for (int k = 0; k < L2; ++k) {
            double2 v = a[k];
            if (s > 0 && k > 0) {
                double2 w = __ldg(tw + s * k); // s k < 2 L2 < L
                if (INV) w.y = -w.y;
                v = cmul(v, w);
            }
            smem[(s * L2 + k) * FFT_R3_COMPS + c] = v;
        }
    }
    __syncthreads();
    if (!live) return;
    // thread m = s: X[k + L2 m] = Z0 + w3^m Z1 + w3^{2m} Z2,  w3 = exp(-+ 2 pi i / 3) = -1/2 -+ i sqrt(3)/2
    constexpr double H = 0.86602540378443864676372317075294; // sqrt(3) / 2
    const double sg = (s == 0) ? 0.0 : ((s == 1) != INV ? -1.0 : 1.0); // sign of the i sqrt(3)/2 (Z1 - Z2) term
#pragma unroll
    for (int k = 0; k < L2; ++k) {
        const double2 z0 = smem[(0 * L2 + k) * FFT_R3_COMPS + c];
        const double2 z1 = smem[(1 * L2 + k) * FFT_R3_COMPS + c];
        const double2 z2 = smem[(2 * L2 + k) * FFT_R3_COMPS + c];
        const double2 t1 = cadd(z1, z2), t2 = csub(z1, z2);
        double2 v;
        if (s == 0) v = cadd(z0, t1);
        else { // z0 - t1 / 2 + sg * i * H * t2,   i * t2 = (-t2.y, t2.x)
            v.x = z0.x - 0.5 * t1.x - sg * H * t2.y;
            v.y = z0.y - 0.5 * t1.y + sg * H * t2.x;
        }
        if (INV) { v.x *= scale; v.y *= scale; }
        data[(s0 + (size_t)(k + L2 * s) * st) * R + r] = v;
    }
}

// ---------------------------------------------------------------------------------------------
// x and y transforms of one z-plane in ONE pass over HBM (rows a2 / a5).  A CTA owns the L x L sites of a plane
// for C consecutive components (16 C-byte segments per site).
//   load   : thread (y, c) copies its x-line into shared memory with L asynchronous 16-byte copies (LDGSTS): they
//            need no registers and no scoreboard entries, so the whole tile is in flight at once -- with plain loads
//            into registers a warp keeps only about seven requests in flight and twelve warps per SM reach half of
//            the copy rate (measured on the memory skeleton of this kernel: 10.7 against 6.2 ms per pass at 32^3);
//   x-lines: the same thread waits for its own copies (no barrier), transforms the line in registers, writes it back;
//   y-lines: after the only barrier thread (x, c) reads its y-line, transforms it and stores it from registers --
//            back in place, or, for the last inverse pass (TOUT), straight into the caller's layout
//            out[component][r] with r = x + L (y + L z): the separate transpose pass disappears.
// Shared layouts (units of 16 bytes; a quarter-warp must hit eight distinct units modulo 8):
//   in place: [y][x][c], row length = L C rounded up to C modulo 8 -> x-line unit = tid + C x, y-line unit = tid + row y
//   TOUT    : [y][c][x] with L + 1 per component: the lanes of the y-lines run over x (coalesced 16 L-byte stores per
//             component), x-line unit = tid + x, y-line units consecutive.
// ---------------------------------------------------------------------------------------------
// components per CTA: 256 / L; at L = 32 NBS_FFT_XY_C (96-byte segments, 99 KB of shared memory, two CTAs per SM)
#ifndef NBS_FFT_XY_C
#define NBS_FFT_XY_C 6
#endif
template <int L>
__host__ __device__ constexpr int fft_xy_comps() { return L >= 32 ? NBS_FFT_XY_C : 256 / L; }
template <int L>
__host__ __device__ constexpr int fft_xy_ctas() { return L >= 32 ? (NBS_FFT_XY_C <= 4 ? 3 : NBS_FFT_XY_C <= 6 ? 2 : 1) : 1; }
template <int L, bool TOUT>
__host__ __device__ constexpr int fft_xy_row() {
    constexpr int C = fft_xy_comps<L>();
    if (TOUT) return C * (L + 1);
    int row = L * C;
    while (row % 8 != C % 8) ++row;
    return row;
}
template <int L, bool TOUT>
constexpr size_t fft_xy_smem_bytes() { return (size_t)L * fft_xy_row<L, TOUT>() * sizeof(double2); }

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}

template <int L, bool INV, bool TOUT>
__global__ void __launch_bounds__(L * fft_xy_comps<L>(), fft_xy_ctas<L>())
k_fft_xy(double2* __restrict__ data, size_t R, size_t Rn, double scale, double2* __restrict__ tout, size_t V) {
    constexpr int C = fft_xy_comps<L>(), NS = L * L, ROW = fft_xy_row<L, TOUT>();
    constexpr int XS = TOUT ? 1 : C, CSTR = TOUT ? L + 1 : 1; // strides of x and of the component inside a row
    extern __shared__ double2 smem[];
    const size_t r0 = (size_t)blockIdx.x * C; // the first Rn components of rows of length R
    const int z = blockIdx.y, tid = threadIdx.x;
    const int nc = (int)((Rn - r0 < (size_t)C) ? (Rn - r0) : (size_t)C);
    double2* plane = data + (size_t)z * NS * R + r0;
    {
        const int y = tid / C, c = tid % C; // x-lines
        if (c < nc) {
            const double2* src = plane + (size_t)y * L * R + c;
            double2* line = smem + y * ROW + c * CSTR;
#pragma unroll
            for (int j = 0; j < L; ++j) cp_async16(line + j * XS, src + (size_t)j * R);
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 0;" ::: "memory"); // this thread's own copies: its line is complete
            double2 a[L];
#pragma unroll
            for (int j = 0; j < L; ++j) a[j] = line[j * XS];
            fft_inreg<L, INV>(a, nullptr);
#pragma unroll
            for (int j = 0; j < L; ++j) line[j * XS] = a[j];
        }
    }
    __syncthreads(); // also: every site of the plane has been read before any is overwritten
    {
        const int x = TOUT ? tid % L : tid / C, c = TOUT ? tid / L : tid % C; // y-lines
        if (c < nc) {
            double2 a[L];
            const double2* src = smem + x * XS + c * CSTR;
#pragma unroll
            for (int j = 0; j < L; ++j) a[j] = src[j * ROW];
            fft_inreg<L, INV>(a, nullptr);
            double2* dst = TOUT ? tout + (r0 + c) * V + (size_t)z * NS + x : plane + (size_t)x * R + c;
            const size_t dstride = TOUT ? (size_t)L : (size_t)L * R;
#pragma unroll
            for (int j = 0; j < L; ++j) {
                double2 v = a[j];
                if (INV) { v.x *= scale; v.y *= scale; }
                dst[(size_t)j * dstride] = v;
            }
        }
    }
}

constexpr int FFT_MAXL = 64;

// Any L (direct O(L^2) DFT); used for lattice sizes that are not powers of two.
template <bool INV>
__global__ void __launch_bounds__(FFT_THREADS)
k_fft_axis_generic(double2* __restrict__ data, size_t R, size_t Rn, int L, int axis, const double2* __restrict__ tw,
                   double scale) {
    size_t r = (size_t)blockIdx.x * FFT_THREADS + threadIdx.x;
    if (r >= Rn) return;
    size_t s0, st;
    line_geometry(L, axis, blockIdx.y, s0, st);
    double2 a[FFT_MAXL], b[FFT_MAXL];
    for (int j = 0; j < L; ++j) a[j] = data[(s0 + j * st) * R + r];
    for (int k = 0; k < L; ++k) {
        double2 acc = make_double2(0.0, 0.0);
        int m = 0;
        for (int j = 0; j < L; ++j) {
            double2 w = __ldg(tw + m);
            if (INV) w.y = -w.y;
            cfma(acc, a[j], w);
            m += k;
            if (m >= L) m -= L;
        }
        b[k] = acc;
    }
    for (int j = 0; j < L; ++j) {
        double2 v = b[j];
        if (INV) { v.x *= scale; v.y *= scale; }
        data[(s0 + j * st) * R + r] = v;
    }
}

// Final layout change: Fr[r][ld] (site-major, the first ncomp components of every row) -> out[comp][r]
// (r fastest), 32x32 tiles.
__global__ void __launch_bounds__(256)
k_transpose_out(const double2* __restrict__ Fr, size_t V, size_t ncomp, size_t ld, double2* __restrict__ out) {
    __shared__ double2 tile[32][33];
    const size_t r0 = (size_t)blockIdx.x * 32, c0 = (size_t)blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int i = ty; i < 32; i += 8) {
        size_t r = r0 + i, c = c0 + tx;
        if (r < V && c < ncomp) tile[i][tx] = Fr[r * ld + c];
    }
    __syncthreads();
    for (int i = ty; i < 32; i += 8) {
        size_t c = c0 + i, r = r0 + tx;
        if (r < V && c < ncomp) out[c * V + r] = tile[tx][i];
    }
}

} // namespace nbs
