// Epilogue of one item of the pipelined product kernel with a pipelined row reader (cf. combine_item, nbs_product.cuh):
// elementary correlators = sums of unit rows in a fixed order (bitwise reproducible), channel correlators = real
// combinations of them (eqs. 2.2-2.3) -> Ft[q][ch][256], mirrored to -q for identical sink baryons
// (reading A11).  Thread et of the ET epilogue threads owns the spin components et + ET m, taken NM at a
// time; the unit rows of the item are read as ONE stream of batches of EG rows, the next batch in flight while the
// current one is summed: the rows come from L2 and the loop is latency-bound (combine_item reads one elementary
// correlator after the other, four rows at a time: 49 ms per launch on its own at 32^3).
#pragma once
#include "nbs_product.cuh"

namespace nbs {

template <int ET, int EG, int NM, bool ALIAS>
__device__ __forceinline__ void combine_item_c(const ProdArgs& a, int ip, size_t q, const double2* __restrict__ scr, int et,
                                               char* s_epi, double osign) {
    constexpr int NMT = 256 / ET;          // components per thread, taken NM at a time (register budget: two batches of EG rows in flight)
    static_assert(NMT % NM == 0, "NM divides the components of a thread");
    Pair3Rec* pr = reinterpret_cast<Pair3Rec*>(s_epi);
    PairChanRec* pcs = reinterpret_cast<PairChanRec*>(s_epi + EPI_PAIR_BYTES);
    {
        const int* src = reinterpret_cast<const int*>(a.pairs + ip);
        if (et < (int)(sizeof(Pair3Rec) / 4)) reinterpret_cast<int*>(pr)[et] = __ldg(src + et);
    }
    named_sync(BAR_EPI, ET);
    const int nelem = pr->nelem, nchan = pr->nchan, swap_mask = pr->swap_mask, nrows = pr->nunits;
    const size_t mq = minus_q(a.L, q);
    const bool mirror = pr->self_swap && mq != q;
    const int src_lane = (et & 0x10) | ((et & 3) << 2) | ((et >> 2) & 3); // a3 <-> a4 inside the 16-lane group
    for (int c0 = 0; c0 < nchan; c0 += EPI_CG) {
        const int nc = min(EPI_CG, nchan - c0);
        {
            const double* src = reinterpret_cast<const double*>(a.pair_chans + pr->chan_begin + c0);
            const int nwords = nc * (int)(sizeof(PairChanRec) / 8);
            for (int i = et; i < nwords; i += ET) reinterpret_cast<double*>(pcs)[i] = __ldg(src + i);
        }
        named_sync(BAR_EPI, ET);
        for (int mh = 0; mh < NMT; mh += NM) {
            auto comp = [&](int m) { return et + ET * (mh + m); };
            // sink swap: F~(-q)_{a2 a1 a3 a4} = - F~(q)_{a1 a2 a3 a4}; component index = ((a1 4 + a2) 4 + a3) 4 + a4
            auto mirror_comp = [&](int m) { const int i = comp(m); return (((i >> 4) & 3) * 4 + (i >> 6)) * 16 + (i & 15); };
            double2 acc[EPI_CG][NM], s[NM];
#pragma unroll
            for (int c = 0; c < EPI_CG; ++c)
#pragma unroll
                for (int m = 0; m < NM; ++m) acc[c][m] = make_double2(0.0, 0.0);
#pragma unroll
            for (int m = 0; m < NM; ++m) s[m] = make_double2(0.0, 0.0);
            int e = 0, eend = pr->elem_unit_begin[1]; // rows [elem_unit_begin[e], elem_unit_begin[e + 1]) belong to elementary correlator e
            auto load = [&](int r0, double2 (&v)[EG][NM]) {
#pragma unroll
                for (int j = 0; j < EG; ++j)
#pragma unroll
                    for (int m = 0; m < NM; ++m)
                        v[j][m] = (r0 + j < nrows) ? __ldcg(scr + (size_t)(r0 + j) * 256 + comp(m)) : make_double2(0.0, 0.0);
            };
            // closes elementary correlator e: source swap (reading A11) by a shuffle, channel coefficients
            auto close_elem = [&]() {
                const bool sw = (swap_mask >> e) & 1;
                double2 ss[NM];
                if (sw) {
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
#pragma unroll
                for (int m = 0; m < NM; ++m) s[m] = make_double2(0.0, 0.0);
                ++e;
                eend = pr->elem_unit_begin[e + 1];
            };
            auto consume = [&](int r0, const double2 (&v)[EG][NM]) {
#pragma unroll
                for (int j = 0; j < EG; ++j) {
                    const int row = r0 + j;
                    if (row < nrows) {
#pragma unroll
                        for (int m = 0; m < NM; ++m) { s[m].x += v[j][m].x; s[m].y += v[j][m].y; }
                        // last row of elementary correlator e (uniform over the threads); one without rows ends at the same row
                        while (row + 1 == eend && e < nelem) close_elem();
                    }
                }
            };
            double2 v0[EG][NM], v1[EG][NM];
            load(0, v0);
            for (int r0 = 0; r0 < nrows; r0 += 2 * EG) {
                load(r0 + EG, v1);
                consume(r0, v0);
                load(r0 + 2 * EG, v0);
                consume(r0 + EG, v1);
            }
#pragma unroll
            for (int c = 0; c < EPI_CG; ++c) {
                if (c < nc) {
                    const int ch = pcs[c].ch - a.ch_begin;
                    if (ch >= 0 && ch < a.nch_out) {
#pragma unroll
                        for (int m = 0; m < NM; ++m) {
                            const double2 val = make_double2(acc[c][m].x * osign, acc[c][m].y * osign); // +-1: sign of a derived block (isospin limit)
                            __stcs(a.Ft + (q * a.nch_out + ch) * 256 + comp(m), val);
                            if (!ALIAS && mirror) __stcs(a.Ft + (mq * a.nch_out + ch) * 256 + mirror_comp(m), make_double2(-val.x, -val.y));
                        }
                    }
                    if (ALIAS && mirror) { // reduced plan of the isospin limit: the mirror may be another channel (PairChanRec::mirror_*)
                        const int mch = pcs[c].mirror_ch - a.ch_begin;
                        if (mch >= 0 && mch < a.nch_out) {
                            const double msg = osign * pcs[c].mirror_sign;
                            const bool msw = pcs[c].mirror_swap != 0;
#pragma unroll
                            for (int m = 0; m < NM; ++m) {
                                const int i = mirror_comp(m), im = msw ? ((i & ~15) | ((i & 3) << 2) | ((i >> 2) & 3)) : i;
                                __stcs(a.Ft + (mq * a.nch_out + mch) * 256 + im, make_double2(acc[c][m].x * msg, acc[c][m].y * msg));
                            }
                        }
                    }
                    // isospin limit, reduced channel list: the u <-> d image of this channel is written from it (nbs_tables.hpp, IsoRelation)
                    const int cha = pcs[c].alias_ch - a.ch_begin;
                    if (ALIAS && pcs[c].alias_ch >= 0 && cha >= 0 && cha < a.nch_out) {
                        const double asg = osign * pcs[c].alias_sign;
                        const bool asw = pcs[c].alias_swap != 0;
                        auto swap34 = [&](int i) { return asw ? ((i & ~15) | ((i & 3) << 2) | ((i >> 2) & 3)) : i; };
#pragma unroll
                        for (int m = 0; m < NM; ++m) {
                            const double2 val = make_double2(acc[c][m].x * asg, acc[c][m].y * asg);
                            __stcs(a.Ft + (q * a.nch_out + cha) * 256 + swap34(comp(m)), val);
                            if (mirror) __stcs(a.Ft + (mq * a.nch_out + cha) * 256 + swap34(mirror_comp(m)), make_double2(-val.x, -val.y));
                        }
                    }
                }
            }
        }
        named_sync(BAR_EPI, ET); // the channel records may be overwritten by the next pass / item
    }
}

} // namespace nbs
