// C-ABI entry points (include/nbs.h).  Host orchestration only; all arithmetic is in the kernels.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "nbs_kernels.cuh"
#include "nbs_product.cuh"
#include "nbs_product_c.cuh"
#include "nbs_probe.cuh"
#include "nbs_tables.hpp"

using namespace nbs;

namespace {

std::string g_create_error = "";

constexpr int NSLOTS_MAX = 2; // time slices in flight (cudaStream overlap)

struct Slice {
    int t = -1;
    const double2* S[3] = {nullptr, nullptr, nullptr}; // u, d, s (device)
    double2* own[3] = {nullptr, nullptr, nullptr};     // library-owned copies for host input
    double2* B = nullptr;  // [V][R] normal blocks, compact rows, x-space then momentum space (in place)
    double2* Be = nullptr; // [V][Re] antisymmetric blocks expanded to full staged blocks (momentum space)
    double2* Ft = nullptr; // [V][nch][256]
    double2* scratch = nullptr;            // [grid][PROD_NBUF][max_pair_units][256] unit results
    unsigned long long* counter = nullptr; // work-item counter of the persistent product kernel
    // in-flight guard: `done` is recorded on the stream of the last call that touched this slot; a call
    // that arrives on another stream first makes its stream wait for it (slices that share a slot serialise)
    cudaEvent_t done = nullptr;
    cudaStream_t last_stream = nullptr;
    bool busy = false;
};

} // namespace

struct nbs_ctx {
    int L = 0, T = 0, device = 0;
    size_t V = 0;
    Plan plan;
    std::string err = "";
    bool cuda_failed = false;
    size_t workspace = 0;
    int nslices = 0;
    Slice slice[NSLOTS_MAX];
    size_t R = 0;  // compact block row length (complex): Plan::row_elems (nbs_tables.hpp)
    size_t Re = 0; // expanded row length: n_asym * SM_BLOCK
    // device tables
    Pair3Rec* d_pairs3 = nullptr;
    Unit3Rec* d_units3 = nullptr;
    Diag3Rec* d_diags3 = nullptr;
    uint2x* d_tab3 = nullptr;
    ChainRec* d_chain = nullptr;
    PairChanRec* d_pair_chans = nullptr;
    int* d_qorder = nullptr;
    int prod_grid = 0;
    // pipelined product kernel (nbs_product_c.cuh): compact antisymmetric blocks staged as they are, no expansion
    bool use_c = false;    // the pipelined kernel is available (program, shared memory) ...
    bool pipelined = false; // ... and selected (nbs_set_pipelined; default: yes when available)
    uint32_t* d_tabc = nullptr;
    Diag3Rec* d_diagsc = nullptr;
    CItem* d_cprog = nullptr;
    CLoad* d_cloads = nullptr;
    int* d_slot_off = nullptr;      // block staged for a slot: its own ...
    int* d_slot_off_iso = nullptr;  // ... or, in the isospin limit, its partner's
    double* d_pair_sign = nullptr;  // all +1
    double* d_pair_sign_iso = nullptr;
    uint32_t c_rec_stride = 0, c_units_bytes = 0;
    size_t c_smem = 0;
    // Isospin limit (d == u), channel relations (nbs_tables.hpp, IsoRelation): a second plan over the channels that are
    // not the u <-> d image of an earlier one; the epilogue writes the images from their originals.  Block rows, FFT
    // and workspace are those of the full plan: only the product stage changes tables.
    struct IsoChannels {
        bool ok = false;
        Plan plan;
        int nderived = 0;
        Pair3Rec* d_pairs3 = nullptr;
        PairChanRec* d_pair_chans = nullptr;
        Unit3Rec* d_units3 = nullptr;
        Diag3Rec* d_diagsc = nullptr;
        uint32_t* d_tabc = nullptr;
        CItem* d_cprog = nullptr;
        CLoad* d_cloads = nullptr;
        int* d_slot_off = nullptr;
        double* d_pair_sign = nullptr;
        uint32_t rec_stride = 0, units_bytes = 0;
        size_t smem = 0;
    } isoch;
    bool iso_relations = true; // nbs_set_channel_relations
    bool direct = false; // nbs_set_direct: eq. 2.4 as a shifted sum in x-space (tiny lattices)
    // Tile-wise plan (BASELINE.json configs[4], 96^3): chosen by nbs_create when the resident
    // workspace does not fit.  A chunk = two sink-spin planes of one baryon for all momenta, [V][2 * SM_PLANE],
    // built on demand (k_blocks in plane-pair mode, forward FFT, expansion) and cached; the product kernel runs
    // once per (sink pair, plane pair of B~1, plane pair of B~2).
    bool tiled = false;
    struct Chunk { double2* buf = nullptr; int slot = -1, pp = -1; long long stamp = 0; };
    std::vector<Chunk> chunks;
    long long chunk_clock = 0, chunk_builds = 0;
    int* d_gather_pp[2] = {nullptr, nullptr};
    int* d_qorder_all = nullptr;  // every momentum, q and -q adjacent
    int* d_qorder_half = nullptr; // the momenta q <= -q
    long long ntasks_half = 0;
    size_t ft_rows = 0;           // rows of Ft per momentum (tile-wise plan: most channels of one sink pair)
    double2* stage_out = nullptr; // tile-wise plan, host output: one channel [256][V]
    long long ntasks = 0;   // entries of d_qorder
    long long nselfconj = 0; // momenta with q == -q
    int* d_baryon_of_slot = nullptr;
    int* d_one_baryon = nullptr; // scratch for nbs_blocks_x
    int2* d_slot_info = nullptr;     // (row offset, block kind) of every slot
    int* d_gather = nullptr;         // expansion map of the antisymmetric slots
    int* d_gather_iso = nullptr;     // the same for the isospin-limit fast path (d == u)
    unsigned dq_mask_iso = 0;
    int2x* d_slot_src = nullptr;     // where the product kernel stages every slot from
    int2* d_one_slot_info = nullptr; // the same for a single baryon (nbs_blocks_x)
    BlockRec* d_brec = nullptr;
    uint16_t* d_blk_out = nullptr; // k_blocks: where a thread's tile goes in the half-row buffer (blocks_out_offsets)
    BTermRec* d_bterm = nullptr;
    double2* d_tw = nullptr;
    unsigned dq_mask = 0;
    unsigned dq_mask_of[NBS_NUM_BARYONS] = {};
    std::vector<void*> allocs;
    long long launches = 0;
    // optional per-stage device timing (nbs_set_timing): events recorded on the launching stream
    bool timing = false;
    struct Pending { int stage; cudaEvent_t a, b; };
    std::vector<Pending> pending;
    std::vector<cudaEvent_t> event_pool;
    double stage_ms[NBS_NUM_STAGES] = {};
    long long stage_calls[NBS_NUM_STAGES] = {};
};

namespace {

int fail(nbs_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}
int cuda_fail(nbs_ctx* c, cudaError_t e, const char* what) {
    if (c) c->cuda_failed = true;
    return fail(c, NBS_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CU(c, call)                                            \
    do {                                                       \
        cudaError_t e_ = (call);                               \
        if (e_ != cudaSuccess) return cuda_fail(c, e_, #call); \
    } while (0)

struct StageTimer { // brackets the launches of one stage with two events on `st`
    nbs_ctx* c; int stage; cudaStream_t st; cudaEvent_t a = nullptr, b = nullptr;
    static cudaEvent_t get(nbs_ctx* c) {
        if (!c->event_pool.empty()) { cudaEvent_t e = c->event_pool.back(); c->event_pool.pop_back(); return e; }
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
        return e;
    }
    StageTimer(nbs_ctx* c_, int stage_, cudaStream_t st_) : c(c_), stage(stage_), st(st_) {
        if (!c->timing) return;
        a = get(c); b = get(c);
        if (!a || !b) { // no event: this stage execution is not timed
            if (a) c->event_pool.push_back(a);
            if (b) c->event_pool.push_back(b);
            a = b = nullptr;
            return;
        }
        cudaEventRecord(a, st);
    }
    ~StageTimer() {
        if (!a) return;
        cudaEventRecord(b, st);
        c->pending.push_back({stage, a, b});
    }
};

template <typename Tp>
int upload(nbs_ctx* c, Tp*& dst, const std::vector<Tp>& src) {
    size_t bytes = std::max<size_t>(src.size(), 1) * sizeof(Tp);
    void* p = nullptr;
    CU(c, cudaMalloc(&p, bytes));
    c->allocs.push_back(p);
    c->workspace += bytes;
    if (!src.empty()) CU(c, cudaMemcpy(p, src.data(), src.size() * sizeof(Tp), cudaMemcpyHostToDevice));
    dst = (Tp*)p;
    return NBS_OK;
}
int dev_alloc(nbs_ctx* c, double2*& dst, size_t ncomplex) {
    void* p = nullptr;
    CU(c, cudaMalloc(&p, ncomplex * sizeof(double2)));
    c->allocs.push_back(p);
    c->workspace += ncomplex * sizeof(double2);
    dst = (double2*)p;
    return NBS_OK;
}

bool fft_r3(int L) { // 3 * 2^k, k = 1..5: the decimation-by-3 kernel
    if (L % 3) return false;
    const int m = L / 3;
    return m == 2 || m == 4 || m == 8 || m == 16 || m == 32;
}

template <int L2, bool INV>
void launch_r3(double2* data, size_t R, size_t Rn, int axis, const double2* tw, double scale, cudaStream_t st) {
    dim3 grid((unsigned)((Rn + FFT_R3_COMPS - 1) / FFT_R3_COMPS), (unsigned)(9 * L2 * L2));
    k_fft_axis_r3<L2, INV><<<grid, dim3(FFT_R3_COMPS, 3), fft_r3_smem_bytes<L2>(), st>>>(data, R, Rn, axis, tw, scale);
}

template <bool INV>
int launch_fft_axis(nbs_ctx* c, double2* data, size_t R, int axis, double scale, cudaStream_t st, size_t Rn = 0) {
    const int L = c->L;
    if (Rn == 0) Rn = R; // Rn: number of (leading) components to transform; R: row length
    if (fft_r3(L)) {
        switch (L / 3) {
        case 2: launch_r3<2, INV>(data, R, Rn, axis, c->d_tw, scale, st); break;
        case 4: launch_r3<4, INV>(data, R, Rn, axis, c->d_tw, scale, st); break;
        case 8: launch_r3<8, INV>(data, R, Rn, axis, c->d_tw, scale, st); break;
        case 16: launch_r3<16, INV>(data, R, Rn, axis, c->d_tw, scale, st); break;
        default: launch_r3<32, INV>(data, R, Rn, axis, c->d_tw, scale, st); break;
        }
        CU(c, cudaGetLastError());
        ++c->launches;
        return NBS_OK;
    }
    dim3 grid((unsigned)((Rn + FFT_THREADS - 1) / FFT_THREADS), (unsigned)(L * L));
    switch (L) {
    case 2: k_fft_axis_pow2<2, INV><<<grid, FFT_THREADS, 0, st>>>(data, R, Rn, axis, c->d_tw, scale); break;
    case 4: k_fft_axis_pow2<4, INV><<<grid, FFT_THREADS, 0, st>>>(data, R, Rn, axis, c->d_tw, scale); break;
    case 8: k_fft_axis_pow2<8, INV><<<grid, FFT_THREADS, 0, st>>>(data, R, Rn, axis, c->d_tw, scale); break;
    case 16: k_fft_axis_pow2<16, INV><<<grid, FFT_THREADS, 0, st>>>(data, R, Rn, axis, c->d_tw, scale); break;
    case 32: k_fft_axis_pow2<32, INV><<<grid, FFT_THREADS, 0, st>>>(data, R, Rn, axis, c->d_tw, scale); break;
    default: k_fft_axis_generic<INV><<<grid, FFT_THREADS, 0, st>>>(data, R, Rn, L, axis, c->d_tw, scale); break;
    }
    CU(c, cudaGetLastError());
    ++c->launches;
    return NBS_OK;
}

template <int L, bool INV, bool TOUT>
int launch_fft_xy(nbs_ctx* c, double2* data, size_t R, size_t Rn, double scale, double2* tout, cudaStream_t st) {
    constexpr int C = fft_xy_comps<L>();
    dim3 grid((unsigned)((Rn + C - 1) / C), (unsigned)L);
    k_fft_xy<L, INV, TOUT><<<grid, L * C, fft_xy_smem_bytes<L, TOUT>(), st>>>(data, R, Rn, scale, tout, c->V);
    CU(c, cudaGetLastError());
    ++c->launches;
    return NBS_OK;
}
template <bool INV, bool TOUT>
int launch_fft_xy_any(nbs_ctx* c, double2* data, size_t R, size_t Rn, double scale, double2* tout, cudaStream_t st) {
    switch (c->L) {
    case 2: return launch_fft_xy<2, INV, TOUT>(c, data, R, Rn, scale, tout, st);
    case 4: return launch_fft_xy<4, INV, TOUT>(c, data, R, Rn, scale, tout, st);
    case 8: return launch_fft_xy<8, INV, TOUT>(c, data, R, Rn, scale, tout, st);
    case 16: return launch_fft_xy<16, INV, TOUT>(c, data, R, Rn, scale, tout, st);
    default: return launch_fft_xy<32, INV, TOUT>(c, data, R, Rn, scale, tout, st);
    }
}
bool fft_fused(const nbs_ctx* c) { return c->L == 2 || c->L == 4 || c->L == 8 || c->L == 16 || c->L == 32; }

// 3-D transform of the first Rn components of data[site][R].  L a power of two <= 32: a z pass at the HBM copy rate,
// then ONE pass for x and y (k_fft_xy: x-lines from HBM into registers, y-lines through shared memory); the last
// inverse pass with `tout` != NULL writes out[comp][r] directly, which saves the transpose pass.  Other L: three
// per-axis passes; tout is ignored and the caller transposes.
int fft3d(nbs_ctx* c, double2* data, size_t R, bool inverse, cudaStream_t st, double2* tout = nullptr, size_t Rn = 0) {
    if (Rn == 0) Rn = R;
    if (fft_fused(c)) {
        const double sz = 1.0 / (double)c->L, sxy = 1.0 / ((double)c->L * c->L);
        int rc = inverse ? launch_fft_axis<true>(c, data, R, 2, sz, st, Rn) : launch_fft_axis<false>(c, data, R, 2, 1.0, st, Rn);
        if (rc) return rc;
        if (!inverse) return launch_fft_xy_any<false, false>(c, data, R, Rn, 1.0, nullptr, st);
        if (tout) return launch_fft_xy_any<true, true>(c, data, R, Rn, sxy, tout, st);
        return launch_fft_xy_any<true, false>(c, data, R, Rn, sxy, nullptr, st);
    }
    for (int axis = 0; axis < 3; ++axis) {
        int rc = inverse ? launch_fft_axis<true>(c, data, R, axis, 1.0 / (double)c->L, st, Rn)
                         : launch_fft_axis<false>(c, data, R, axis, 1.0, st, Rn);
        if (rc) return rc;
    }
    return NBS_OK;
}

int launch_blocks(nbs_ctx* c, const Slice& s, const int* d_list, const int2* d_info, int nslots, unsigned dq_mask,
                  double2* out, size_t row_stride, cudaStream_t st, int pp = -1) {
    int ndq = 0;
    for (int b = 0; b < 9; ++b) ndq += (dq_mask >> b) & 1u;
    if (nslots > BLOCKS_MAX_SLOTS) return fail(c, NBS_EINVAL, "too many block slots");
    k_blocks<<<(unsigned)c->V, BLOCKS_THREADS, blocks_smem_bytes(ndq), st>>>(s.S[0], s.S[1], s.S[2], d_list, nslots, dq_mask,
                                                                          c->d_brec, c->d_bterm, d_info, c->d_blk_out, out, row_stride, pp);
    CU(c, cudaGetLastError());
    ++c->launches;
    return NBS_OK;
}

// In-flight guard of a workspace slot (include/nbs.h, nbs_num_slots): order this call after whatever the slot
// was last used for when that happened on another stream.
int slot_acquire(nbs_ctx* c, Slice& sl, cudaStream_t st) {
    if (sl.busy && sl.last_stream != st) CU(c, cudaStreamWaitEvent(st, sl.done, 0));
    return NBS_OK;
}
int slot_release(nbs_ctx* c, Slice& sl, cudaStream_t st) {
    CU(c, cudaEventRecord(sl.done, st));
    sl.last_stream = st;
    sl.busy = true;
    return NBS_OK;
}


// ---- tile-wise plan ---------------------------------------------------------------------------
// Chunk (slot, pp) of the loaded slice: k_blocks in plane-pair mode writes the two sink-spin planes (staged for a
// block without antisymmetry, compact for an antisymmetric one) into rows of 2 * SM_PLANE entries, the forward
// FFT transforms them in place, k_expand_chunk restores the mirror entries of an antisymmetric block in place.
int get_chunk(nbs_ctx* c, Slice& sl, int slot, int pp, int protect, cudaStream_t st, int* index) {
    for (size_t i = 0; i < c->chunks.size(); ++i)
        if (c->chunks[i].slot == slot && c->chunks[i].pp == pp) {
            c->chunks[i].stamp = ++c->chunk_clock;
            *index = (int)i;
            return NBS_OK;
        }
    int victim = -1;
    for (size_t i = 0; i < c->chunks.size(); ++i) {
        if ((int)i == protect) continue;
        if (victim < 0 || c->chunks[i].slot < 0 ||
            (c->chunks[victim].slot >= 0 && c->chunks[i].stamp < c->chunks[victim].stamp))
            victim = (int)i;
        if (c->chunks[victim].slot < 0) break;
    }
    nbs_ctx::Chunk& ck = c->chunks[victim];
    const int baryon = c->plan.baryons[slot], kind = c->plan.slot_kind[slot];
    const size_t R = 2 * SM_PLANE;
    int rc;
    {
        StageTimer tm(c, NBS_STAGE_BLOCKS, st);
        rc = launch_blocks(c, sl, c->d_one_baryon + baryon, c->d_one_slot_info + baryon, 1, c->dq_mask_of[baryon], ck.buf, R, st, pp);
        if (rc) return rc;
    }
    {
        StageTimer tm(c, NBS_STAGE_FFT_FWD, st);
        rc = fft3d(c, ck.buf, R, false, st, nullptr, kind == BK_FULL ? R : (size_t)(2 * AS_PLANE));
        if (rc) return rc;
        if (kind != BK_FULL) {
            k_expand_chunk<<<(unsigned)c->V, 256, 0, st>>>(ck.buf, c->d_gather_pp[kind - 1]);
            CU(c, cudaGetLastError());
            ++c->launches;
        }
    }
    ck.slot = slot; ck.pp = pp; ck.stamp = ++c->chunk_clock;
    ++c->chunk_builds;
    *index = victim;
    return NBS_OK;
}

// nbs_correlator with the tile-wise plan: sink pair by sink pair (in chain order, so that consecutive pairs share
// chunks), each as up to four launches of the product kernel, one per (plane pair of B~1, plane pair of B~2);
// then the inverse FFT of the pair's channels and their final layout in the caller's buffer.
int correlator_tiled(nbs_ctx* c, Slice& sl, int ch_begin, int ch_end, void* out, int memloc, cudaStream_t st) {
    const Plan& P = c->plan;
    const size_t chan_elems = 256 * c->V;
    if (memloc == NBS_MEM_HOST && !c->stage_out) {
        int rc = dev_alloc(c, c->stage_out, chan_elems);
        if (rc) return rc;
    }
    for (int ci = 0; ci < P.chain_full_n; ++ci) {
        const int ip = P.chain[ci].pair;
        const Pair3Rec& pr = P.pairs3[ip];
        bool wanted = false;
        for (int k = 0; k < pr.nchan; ++k) {
            const int ch = P.pair_chans[pr.chan_begin + k].ch;
            wanted = wanted || (ch >= ch_begin && ch < ch_end);
        }
        if (!wanted) continue;
        // plane-pair tiles; for identical sink baryons (1,0) follows from (0,1) by the sink swap (reading A11)
        static const int tiles[4][2] = {{0, 0}, {0, 1}, {1, 1}, {1, 0}};
        const int ntiles = pr.self_swap ? 3 : 4;
        for (int it = 0; it < ntiles; ++it) {
            const int ti = tiles[it][0], tj = tiles[it][1];
            int i1 = -1, i2 = -1;
            int rc = get_chunk(c, sl, pr.slot1, ti, -1, st, &i1);
            if (rc) return rc;
            rc = get_chunk(c, sl, pr.slot2, tj, i1, st, &i2);
            if (rc) return rc;
            StageTimer tm(c, NBS_STAGE_PRODUCT, st);
            CU(c, cudaMemsetAsync(sl.counter, 0, sizeof(unsigned long long), st));
            ProdArgs pa;
            pa.Bc = nullptr; pa.Rc = 0; pa.Be = nullptr; pa.Re = 0; pa.L = c->L;
            pa.slot_src = reinterpret_cast<const int2*>(c->d_slot_src);
            pa.chain_full_n = P.chain_full_n; pa.chain_half_n = P.chain_half_n;
            const bool half = pr.self_swap && ti == tj; // the momenta q <= -q, mirrored to -q by the epilogue
            pa.ntasks = half ? c->ntasks_half : (long long)c->V;
            pa.qorder = half ? c->d_qorder_half : c->d_qorder_all;
            pa.direct = 0;
            pa.pairs = c->d_pairs3; pa.units = c->d_units3; pa.diags = c->d_diags3;
            pa.tab = reinterpret_cast<const uint2*>(c->d_tab3);
            pa.pair_chans = c->d_pair_chans; pa.chain = c->d_chain;
            pa.scratch = sl.scratch; pa.max_pair_units = P.max_pair_units;
            pa.Ft = sl.Ft; pa.ch_begin = 0; pa.nch_out = pr.nchan;
            pa.counter = sl.counter;
            pa.c1 = c->chunks[i1].buf; pa.c2 = c->chunks[i2].buf;
            pa.tile_i = ti; pa.tile_j = tj; pa.chain_base = P.chain_single_begin + ip;
            unsigned grid = (unsigned)std::min<long long>(c->prod_grid, pa.ntasks);
            k_product_t<true><<<grid, PROD_THREADS, PROD_SMEM, st>>>(pa);
            CU(c, cudaGetLastError());
            ++c->launches;
        }
        const size_t ld = (size_t)pr.nchan * 256;
        {
            StageTimer tm(c, NBS_STAGE_FFT_INV, st);
            int rc = fft3d(c, sl.Ft, ld, true, st);
            if (rc) return rc;
        }
        StageTimer tm(c, NBS_STAGE_OUTPUT, st);
        for (int k = 0; k < pr.nchan; ++k) {
            const PairChanRec& pc = P.pair_chans[pr.chan_begin + k];
            if (pc.ch < ch_begin || pc.ch >= ch_end) continue;
            double2* dst = memloc == NBS_MEM_HOST ? c->stage_out : (double2*)out + (size_t)(pc.ch - ch_begin) * chan_elems;
            dim3 tg((unsigned)((c->V + 31) / 32), 8);
            k_transpose_out<<<tg, 256, 0, st>>>(sl.Ft + (size_t)pc.local * 256, c->V, 256, ld, dst);
            CU(c, cudaGetLastError());
            ++c->launches;
            if (memloc == NBS_MEM_HOST)
                CU(c, cudaMemcpyAsync((double2*)out + (size_t)(pc.ch - ch_begin) * chan_elems, dst, chan_elems * sizeof(double2),
                                      cudaMemcpyDeviceToHost, st));
        }
    }
    return NBS_OK;
}

} // namespace

extern "C" {

int nbs_std_channels(nbs_channel* out, int cap) {
    std::vector<nbs_channel> ch = standard_channels();
    for (int i = 0; i < (int)ch.size() && i < cap; ++i) out[i] = ch[i];
    return (int)ch.size();
}

int nbs_diagram_stats(const nbs_channel* ch, int* K, int* sign, int cap, long long* literal_terms) {
    if (!ch) return NBS_EINVAL;
    std::vector<DiagramInfo> d;
    std::string err = channel_diagrams(*ch, d);
    if (!err.empty()) { g_create_error = err; return NBS_EINVAL; }
    for (int i = 0; i < (int)d.size() && i < cap; ++i) {
        if (K) K[i] = d[i].K;
        if (sign) sign[i] = d[i].sign;
    }
    if (literal_terms) *literal_terms = (long long)d.size() * 576; // (N_c! N_alpha)^B
    return (int)d.size();
}

int nbs_iso_relations(const nbs_channel* ch, int nch, int* from, int* sign, int* swap34, int cap) {
    std::vector<nbs_channel> chans = ch ? std::vector<nbs_channel>(ch, ch + nch) : standard_channels();
    for (auto& x : chans)
        for (int b : {x.b1, x.b2, x.b3, x.b4})
            if (b < 0 || b >= NBS_NUM_BARYONS) return NBS_EINVAL;
    const std::vector<IsoRelation> rel = iso_channel_relations(chans);
    for (size_t i = 0; i < rel.size() && (int)i < cap; ++i) {
        if (from) from[i] = rel[i].from;
        if (sign) sign[i] = rel[i].sign;
        if (swap34) swap34[i] = rel[i].swap34;
    }
    return (int)rel.size();
}

static int plan_selfcheck(const Plan& P);

// The reduced plan of the isospin limit (build_iso_channels): the channels that are no u <-> d image, with the mirror
// relation of conjugate sink pairs switched on.  Returns false if the list has neither an image nor a conjugate pair.
static bool reduced_iso_plan(const std::vector<nbs_channel>& chans, Plan& rp, std::vector<int>& orig, std::string& err) {
    const std::vector<IsoRelation> rel = iso_channel_relations(chans);
    std::vector<nbs_channel> red;
    orig.clear();
    for (size_t i = 0; i < rel.size(); ++i)
        if (rel[i].from < 0) { red.push_back(chans[i]); orig.push_back((int)i); }
    std::vector<char> carries(red.size(), 0); // channels that carry an image to write take no part in the mirror relation
    for (size_t i = 0; i < rel.size(); ++i)
        if (rel[i].from >= 0)
            for (size_t k = 0; k < orig.size(); ++k)
                if (orig[k] == rel[i].from) carries[k] = 1;
    err = build_plan(red, rp, UNIT_SPLIT_STEPS_DEFAULT, UNIT_COST_MAX_DEFAULT, &carries);
    if (!err.empty()) return true;
    bool conj = false;
    for (auto& pr : rp.pairs3) conj = conj || pr.self_swap == 2;
    return conj || red.size() < chans.size();
}

int nbs_plan_selfcheck(const nbs_channel* ch, int nch) {
    // Host-side bounds check of everything the kernels index with table data (compute-sanitizer is not available on
    // the target pool): returns 0, or the negative number of the first violated invariant.
    std::vector<nbs_channel> chans = ch ? std::vector<nbs_channel>(ch, ch + nch) : standard_channels();
    for (auto& x : chans)
        for (int b : {x.b1, x.b2, x.b3, x.b4})
            if (b < 0 || b >= NBS_NUM_BARYONS) return NBS_EINVAL;
    Plan P;
    std::string err = build_plan(chans, P);
    if (!err.empty()) { g_create_error = err; return NBS_EINVAL; }
    int rc = plan_selfcheck(P);
    if (rc) return rc;
    // the reduced plan of the isospin limit: the same invariants (1000 is subtracted from the check number), and the
    // mirror relation of its conjugate sink pairs: an involution inside the pair, signs +-1, no channel that carries an image
    Plan R;
    std::vector<int> orig;
    if (!reduced_iso_plan(chans, R, orig, err)) return 0;
    if (!err.empty()) { g_create_error = err; return -1150; }
    rc = plan_selfcheck(R);
    if (rc) return rc - 1000;
    for (auto& pr : R.pairs3)
        for (int k = 0; k < pr.nchan; ++k) {
            const PairChanRec& pc = R.pair_chans[pr.chan_begin + k];
            if (pr.self_swap != 2) {
                if (pc.mirror_ch != pc.ch || pc.mirror_swap != 0 || pc.mirror_sign != -1.0) return -1151;
                continue;
            }
            const PairChanRec* m = nullptr;
            for (int j = 0; j < pr.nchan; ++j)
                if (R.pair_chans[pr.chan_begin + j].ch == pc.mirror_ch) m = &R.pair_chans[pr.chan_begin + j];
            if (!m) return -1152;                                   // the mirror channel belongs to the same sink pair
            if (m->mirror_ch != pc.ch || m->mirror_swap != pc.mirror_swap || m->mirror_sign != pc.mirror_sign) return -1153; // involution
            if (pc.mirror_sign != 1.0 && pc.mirror_sign != -1.0) return -1154;
            if (R.baryons[pr.slot1] == R.baryons[pr.slot2]) return -1155;
        }
    return 0;
}

static int plan_selfcheck(const Plan& P) {
    const size_t ntab = P.tab3.size();
    for (auto& w : P.tab3) // 1: gather offsets are 16-byte aligned positions inside a staged block
        if (w.x % 16 || w.y % 16 || w.x >= BLOCK_BYTES || w.y >= BLOCK_BYTES) return -101;
    for (auto& d : P.diags3) { // 2: a diagram's tables, one k-step past its range (software pipeline), lie inside tab3
        const size_t rowsA = 8, stepA = 4 * rowsA * d.nwA, stepB4 = 4 * 4 * d.nwB, stepB8 = 4 * 8 * d.nwB;
        if (d.send <= d.sbeg || d.send > (d.K + 3) / 4) return -102;
        if (d.offA + (size_t)(d.send + 1) * std::max<size_t>(stepA, 4 * 8 * 4) > ntab) return -103;
        if (d.offB + (size_t)(d.send + 1) * std::max(stepB4, stepB8) > ntab) return -104;
        if (d.offA % 2 || d.offB % 2) return -105; // 16-byte aligned tables (uint4 reads)
    }
    if (P.max_pair_units > MAX_PAIR_UNITS) return -106;
    if (P.diagsc.size() != P.diags3.size()) return -130;
    {   // 5: compact gather tables and the program of the pipelined kernel
        const size_t ntabc = P.tabc.size();
        for (uint32_t w : P.tabc) // offsets inside one plane, 16-byte aligned (the kind of the block is checked per unit below)
            if ((w & 0xfu) || ((w >> 16) & 0xfu) || (w & 0x7ff0u) >= PLANE_BYTES || ((w >> 16) & 0x7ff0u) >= PLANE_BYTES) return -131;
        for (size_t i = 0; i < P.diagsc.size(); ++i) {
            const Diag3Rec &d = P.diagsc[i], &o = P.diags3[i];
            if (d.sbeg != o.sbeg || d.send != o.send || d.nwA != o.nwA || d.nwB != o.nwB || d.K != o.K) return -132;
            if (d.offA % 4 || d.offB % 4) return -135;
        }
        for (auto& pr : P.pairs3) // table extents with the register pipeline's look-ahead, by class of the unit
            for (int u = 0; u < pr.nunits; ++u) {
                const Unit3Rec& ur = P.units3[pr.unit_begin + u];
                const int k1 = P.slot_kind[pr.slot1], k2 = P.slot_kind[pr.slot2];
                for (int di = ur.diag_begin; di < ur.diag_end; ++di) {
                    const Diag3Rec& d = P.diagsc[pr.diag_begin + di];
                    const size_t steps = (size_t)d.send + C_TAB_LOOKAHEAD;
                    const size_t wordsA = ur.cls < 2 ? 16 * (size_t)d.nwA : 64, wordsB = ur.cls < 2 ? 16 * (size_t)d.nwB : 16;
                    if (d.offA + steps * wordsA > ntabc) return -133;
                    if (d.offB + steps * wordsB > ntabc) return -134;
                    // the words really used stay inside a plane of the block they address
                    const int kA = ur.cls == 3 ? k2 : k1, kB = ur.cls == 3 ? k1 : k2;
                    for (size_t x = (size_t)d.sbeg * wordsA; x < (size_t)d.send * wordsA; ++x) {
                        const uint32_t w = P.tabc[d.offA + x];
                        if ((w & 0x7ff0u) >= (uint32_t)plane_elems(kA) * 16u || ((w >> 16) & 0x7ff0u) >= (uint32_t)plane_elems(kA) * 16u) return -148;
                    }
                    for (size_t x = (size_t)d.sbeg * wordsB; x < (size_t)d.send * wordsB; ++x) {
                        const uint32_t w = P.tabc[d.offB + x];
                        if ((w & 0x7ff0u) >= (uint32_t)plane_elems(kB) * 16u || ((w >> 16) & 0x7ff0u) >= (uint32_t)plane_elems(kB) * 16u) return -149;
                    }
                }
            }
        if (P.cprog_ok) {
            if ((int)P.cprog.size() != P.chain_full_n + P.chain_half_n || (int)P.cprog.size() < C_NREC) return -136;
            std::vector<int> fresh(C_NSLOT, 0), loaded(C_NSLOT, 0);
            // half slots (nbs_tables.hpp) covered by a block of `kind` whose first slot starts at byte offset `off`
            auto halves = [&](uint32_t off, int kind, unsigned& mask) {
                mask = 0;
                if (off % C_HALF_BYTES) return false;
                const int h = (int)(off / C_HALF_BYTES);
                if (kind == BK_FULL) { if (h % 4) return false; mask = 0xfu << h; }
                else { if (h % 4 > 1) return false; mask = (1u << h) | (1u << (h + 2)); }
                return h < 2 * C_NSLOT && (mask >> (2 * C_NSLOT)) == 0;
            };
            auto slot_of_off = [&](uint32_t off) { const int h = (int)(off / C_HALF_BYTES); return (h / 4) * 2 + (h % 4); };
            for (size_t i = 0; i < P.cprog.size(); ++i) {
                const CItem& it = P.cprog[i];
                const Pair3Rec& pr = P.pairs3[it.pair];
                unsigned m1, m2;
                if (!halves(it.off1, P.slot_kind[pr.slot1], m1) || !halves(it.off2, P.slot_kind[pr.slot2], m2)) return -137;
                if (m1 & m2) return -139; // the two blocks of an item do not overlap
                if (it.ps1 != (uint32_t)plane_elems(P.slot_kind[pr.slot1]) * 16u || it.ps2 != (uint32_t)plane_elems(P.slot_kind[pr.slot2]) * 16u) return -140;
                if (it.rel_begin > it.rel_end || it.rel_end > (int)P.cloads.size()) return -141;
                for (int side = 0; side < 2; ++side) {
                    const int w = (it.flags >> (3 * side)) & 7;
                    if (w > C_NSLOT) return -142;
                    if (w && w - 1 != slot_of_off(side ? it.off2 : it.off1)) return -143;
                    if (w) ++fresh[w - 1];
                }
            }
            for (auto& ld : P.cloads) {
                if ((ld.src & 255) >= (int)P.baryons.size() || ld.bar < 0 || ld.bar >= C_NSLOT) return -144;
                unsigned m;
                if (!halves(ld.dst, P.slot_kind[ld.src & 255], m) || slot_of_off(ld.dst) != ld.bar) return -145;
                if (ld.bytes != (uint32_t)block_elems(P.slot_kind[ld.src & 255]) * 16u || ld.bytes % 64) return -146;
                ++loaded[ld.bar];
            }
            for (int s = 0; s < C_NSLOT; ++s)
                if (fresh[s] != loaded[s]) return -147; // every load is waited for by exactly one item (barrier phases stay in step)
        }
    }
    for (auto& pr : P.pairs3) {
        if (pr.nunits < 1 || pr.nunits > MAX_PAIR_UNITS || pr.ndiags > MAX_PAIR_DIAGS || pr.nelem > MAX_PAIR_ELEMS) return -107;
        if (pr.unit_begin + pr.nunits > (int)P.units3.size() || pr.diag_begin + pr.ndiags > (int)P.diags3.size()) return -108;
        if (pr.slot1 < 0 || pr.slot1 >= (int)P.baryons.size() || pr.slot2 < 0 || pr.slot2 >= (int)P.baryons.size()) return -109;
        std::vector<char> seen(pr.nunits, 0);
        for (int u = 0; u < pr.nunits; ++u) {
            const Unit3Rec& ur = P.units3[pr.unit_begin + u];
            if (ur.diag_begin < 0 || ur.diag_end > pr.ndiags || ur.diag_begin >= ur.diag_end) return -110;
            if (ur.slot < 0 || ur.slot >= pr.nunits || seen[ur.slot] || ur.cls < 0 || ur.cls > 3) return -111;
            seen[ur.slot] = 1; // every scratch row written by exactly one unit
        }
        for (int e = 0; e < MAX_PAIR_ELEMS; ++e)
            if (pr.elem_unit_begin[e] > pr.elem_unit_begin[e + 1] || pr.elem_unit_begin[e + 1] > pr.nunits) return -112;
        if (pr.chan_begin + pr.nchan > (int)P.pair_chans.size()) return -113;
        for (int k = 0; k < pr.nchan; ++k) {
            const PairChanRec& pc = P.pair_chans[pr.chan_begin + k];
            if (pc.ch < 0 || pc.ch >= (int)P.channels.size() || pc.local != k) return -114;
        }
    }
    if ((int)P.chain.size() != P.chain_full_n + P.chain_half_n + (int)P.pairs3.size()) return -115;
    for (auto& cr : P.chain) {
        if (cr.pair < 0 || cr.pair >= (int)P.pairs3.size()) return -116;
        const Pair3Rec& pr = P.pairs3[cr.pair];
        if (cr.nunits != pr.nunits || cr.unit_begin != pr.unit_begin || cr.ndiags != pr.ndiags || cr.diag_begin != pr.diag_begin) return -117;
        const size_t lim1 = cr.buf1 ? (size_t)P.n_asym * SM_BLOCK : (size_t)P.row_elems;
        const size_t lim2 = cr.buf2 ? (size_t)P.n_asym * SM_BLOCK : (size_t)P.row_elems;
        if ((size_t)cr.off1 + SM_BLOCK > lim1 || (size_t)cr.off2 + SM_BLOCK > lim2) return -118;
    }
    for (int i = 0; i < P.chain_full_n + P.chain_half_n; ++i) { // 3: a reused staged block really is the one staged before
        if (i == 0 || i == P.chain_full_n) { if (!P.chain[i].load1 || !P.chain[i].load2) return -119; continue; }
        const Pair3Rec &a = P.pairs3[P.chain[i - 1].pair], &b = P.pairs3[P.chain[i].pair];
        if ((!P.chain[i].load1 && a.slot1 != b.slot1) || (!P.chain[i].load2 && a.slot2 != b.slot2)) return -120;
    }
    for (size_t j = 0; j < P.gather.size(); ++j) // 4: expansion maps stay inside the compact row / chunk
        if (P.gather[j] >= 0 && (size_t)(P.gather[j] & 0x3fffffff) >= (size_t)P.row_elems) return -121;
    for (size_t j = 0; j < P.gather_iso.size(); ++j)
        if (P.gather_iso[j] >= 0 && (size_t)(P.gather_iso[j] & 0x3fffffff) >= (size_t)P.row_elems_iso) return -122;
    for (int k = 0; k < 2; ++k) {
        if (P.gather_pp[k].size() != (size_t)(2 * SM_PLANE)) return -123;
        for (int g : P.gather_pp[k])
            if (g >= 0 && (g & 0x3fffffff) >= 2 * AS_PLANE) return -124;
    }
    if ((size_t)P.row_elems != (size_t)P.slot_off.back() + block_elems(P.slot_kind.back())) return -125;
    return NBS_OK;
}

// Second plan for the isospin limit: the channels that are not the u <-> d image of an earlier channel of the list
// (nbs_tables.hpp, iso_channel_relations).  Its tables address the block rows of the FULL plan (what k_blocks and the
// forward FFT write when d == u: the blocks of p, Sigma+, Xi0 stand in for n, Sigma-, Xi-), its channel records
// carry the numbers of the full list and the image each of them has to be copied to.  Not available -> isoch.ok stays
// false and the isospin limit runs the full plan (same results).
static int build_iso_channels(nbs_ctx* c, size_t smem_optin) {
    const std::vector<IsoRelation> rel = iso_channel_relations(c->plan.channels);
    nbs_ctx::IsoChannels& ic = c->isoch;
    ic.nderived = 0;
    for (auto& r : rel) ic.nderived += r.from >= 0;
    Plan& rp = ic.plan;
    std::vector<int> orig;
    std::string err;
    if (!reduced_iso_plan(c->plan.channels, rp, orig, err)) return NBS_OK;
    if (!err.empty() || !rp.cprog_ok || rp.max_pair_units > c->plan.max_pair_units || rp.baryons.size() >= 256) return NBS_OK;
    ic.units_bytes = (uint32_t)rp.max_pair_units * (uint32_t)sizeof(Unit3Rec);
    ic.rec_stride = C_ITEM_BYTES + ic.units_bytes + (uint32_t)rp.max_pair_diags * (uint32_t)sizeof(Diag3Rec);
    ic.smem = cprod_smem_bytes(ic.rec_stride);
    if (ic.smem > smem_optin) return NBS_OK;
    for (auto& pc : rp.pair_chans) { pc.ch = orig[pc.ch]; pc.mirror_ch = orig[pc.mirror_ch]; } // channel numbers of the full list
    for (size_t i = 0; i < rel.size(); ++i) {
        if (rel[i].from < 0) continue;
        bool found = false;
        for (auto& pc : rp.pair_chans)
            if (pc.ch == rel[i].from) { pc.alias_ch = (int)i; pc.alias_sign = (double)rel[i].sign; pc.alias_swap = rel[i].swap34; found = true; }
        if (!found) return NBS_OK; // the original has no record (cannot happen for a valid channel): keep the full plan
    }
    // blocks are staged from the rows of the full plan: a derived baryon from its partner's block, with its sign
    std::vector<int> off, sgn;
    for (int b : rp.baryons) {
        int fs = -1;
        for (size_t s = 0; s < c->plan.baryons.size(); ++s)
            if (c->plan.baryons[s] == b) fs = (int)s;
        if (fs < 0) return NBS_OK;
        off.push_back(c->plan.slot_off[c->plan.slot_partner_iso[fs]]);
        sgn.push_back(c->plan.slot_sign_iso[fs]);
    }
    std::vector<double> psg;
    for (auto& pr : rp.pairs3) psg.push_back((double)(sgn[pr.slot1] * sgn[pr.slot2]));
    int rc;
    if ((rc = upload(c, ic.d_pairs3, rp.pairs3)) || (rc = upload(c, ic.d_pair_chans, rp.pair_chans)) ||
        (rc = upload(c, ic.d_units3, rp.units3)) || (rc = upload(c, ic.d_diagsc, rp.diagsc)) || (rc = upload(c, ic.d_tabc, rp.tabc)) ||
        (rc = upload(c, ic.d_cprog, rp.cprog)) || (rc = upload(c, ic.d_cloads, rp.cloads)) || (rc = upload(c, ic.d_slot_off, off)) ||
        (rc = upload(c, ic.d_pair_sign, psg)))
        return rc;
    ic.ok = true;
    return NBS_OK;
}

int nbs_set_channel_relations(nbs_ctx* c, int enable) {
    if (!c) return NBS_EINVAL;
    if (enable == -2) { // query: sink pairs contracted for half of the momenta thanks to the relations
        int n = 0;
        if (c->isoch.ok && c->iso_relations)
            for (auto& pr : c->isoch.plan.pairs3) n += pr.self_swap == 2;
        return n;
    }
    if (enable < 0) return (c->isoch.ok && c->iso_relations) ? c->isoch.nderived : 0; // query
    c->iso_relations = enable != 0;
    return NBS_OK;
}

int nbs_create(nbs_ctx** out, int L, int T, const nbs_channel* ch, int nch, int device, size_t budget) {
    if (!out) return fail(nullptr, NBS_EINVAL, "out is NULL");
    *out = nullptr;
    if (L < 2 || (L > FFT_MAXL && !fft_r3(L)))
        return fail(nullptr, NBS_EINVAL, "L must be in [2, 64] or 3 * 2^k <= 96");
    if (T < 1) return fail(nullptr, NBS_EINVAL, "T must be >= 1");
    if (ch && nch < 1) return fail(nullptr, NBS_EINVAL, "nch must be >= 1");
    std::vector<nbs_channel> chans = ch ? std::vector<nbs_channel>(ch, ch + nch) : standard_channels();
    nbs_ctx* c = new nbs_ctx();
#if defined(NBS_UNIT_SPLIT) && defined(NBS_UNIT_COST)
    std::string err = build_plan(chans, c->plan, NBS_UNIT_SPLIT, NBS_UNIT_COST);
#else
    std::string err = build_plan(chans, c->plan);
#endif
    if (!err.empty()) { delete c; return fail(nullptr, NBS_EINVAL, err); }
    c->L = L; c->T = T; c->device = device;
    c->V = (size_t)L * L * L;
    c->R = (size_t)c->plan.row_elems;
    c->Re = (size_t)c->plan.n_asym * SM_BLOCK;

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || device < 0 || device >= ndev) {
        std::string msg = e != cudaSuccess ? std::string("no usable CUDA device: ") + cudaGetErrorString(e)
                                           : "device ordinal out of range";
        delete c;
        return fail(nullptr, NBS_ECUDA, msg);
    }
#define CUC(call)                                                                 \
    do {                                                                          \
        int rc_ = (call);                                                         \
        if (rc_ != NBS_OK) { g_create_error = c->err; nbs_destroy(c); return rc_; } \
    } while (0)
#define CUX(call)                                                                                        \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) { g_create_error = std::string(#call) + ": " + cudaGetErrorString(e_); nbs_destroy(c); return NBS_ECUDA; } \
    } while (0)
    CUX(cudaSetDevice(device));

    // block-construction descriptors for all baryon ids
    std::vector<BlockRec> brec(NBS_NUM_BARYONS);
    std::vector<BTermRec> bterm;
    for (int b = 0; b < NBS_NUM_BARYONS; ++b) {
        brec[b].term_begin = (int)bterm.size();
        for (auto& t : block_terms(b)) {
            BTermRec r;
            r.coef = t.coef; r.dq = t.f0 * 3 + t.f1; r.f2 = t.f2;
            r.p0 = t.perm[0]; r.p1 = t.perm[1]; r.p2 = t.perm[2]; r.pad = 0;
            bterm.push_back(r);
            c->dq_mask_of[b] |= 1u << r.dq;
        }
        brec[b].term_end = (int)bterm.size();
    }
    for (int b : c->plan.baryons) c->dq_mask |= c->dq_mask_of[b];
    for (int i = 0; i < c->plan.n_slots_iso; ++i) c->dq_mask_iso |= c->dq_mask_of[c->plan.baryons[i]];
    std::vector<double2> tw(L);
    for (int m = 0; m < L; ++m) {
        long double ang = -2.0L * 3.141592653589793238462643383279502884L * m / L;
        tw[m] = make_double2((double)cosl(ang), (double)sinl(ang));
    }
    CUC(upload(c, c->d_pairs3, c->plan.pairs3));
    CUC(upload(c, c->d_units3, c->plan.units3));
    CUC(upload(c, c->d_diags3, c->plan.diags3));
    CUC(upload(c, c->d_tab3, c->plan.tab3));
    CUC(upload(c, c->d_chain, c->plan.chain));
    CUC(upload(c, c->d_pair_chans, c->plan.pair_chans));
    {
        // momenta ordered so that q and -q are adjacent (their blocks are shared through L2)
        std::vector<int> qorder;
        std::vector<char> seen(c->V, 0);
        auto neg = [&](size_t q) {
            size_t x = q % L, y = (q / L) % L, z = q / ((size_t)L * L);
            x = x ? L - x : 0; y = y ? L - y : 0; z = z ? L - z : 0;
            return x + (size_t)L * (y + (size_t)L * z);
        };
        // if every sink pair has identical baryons the momenta q > -q have nothing to compute
        const bool skip_upper = c->plan.chain_half_n == 0;
        for (size_t q = 0; q < c->V; ++q) {
            if (seen[q]) continue;
            qorder.push_back((int)q); seen[q] = 1;
            size_t m = neg(q);
            if (!seen[m]) { if (!skip_upper) qorder.push_back((int)m); seen[m] = 1; }
        }
        c->ntasks = (long long)qorder.size();
        c->nselfconj = 0;
        for (size_t q = 0; q < c->V; ++q) c->nselfconj += neg(q) == q;
        CUC(upload(c, c->d_qorder, qorder));
        std::vector<int> qall, qhalf;
        std::fill(seen.begin(), seen.end(), 0);
        for (size_t q = 0; q < c->V; ++q) {
            if (seen[q]) continue;
            const size_t m = neg(q);
            qall.push_back((int)q); qhalf.push_back((int)q); seen[q] = 1;
            if (!seen[m]) { qall.push_back((int)m); seen[m] = 1; }
        }
        c->ntasks_half = (long long)qhalf.size();
        CUC(upload(c, c->d_qorder_all, qall));
        CUC(upload(c, c->d_qorder_half, qhalf));
        CUC(upload(c, c->d_gather_pp[0], c->plan.gather_pp[0]));
        CUC(upload(c, c->d_gather_pp[1], c->plan.gather_pp[1]));
    }
    size_t smem_optin = 0;
    {
        cudaDeviceProp prop;
        CUX(cudaGetDeviceProperties(&prop, device));
        if ((size_t)prop.sharedMemPerBlockOptin < PROD_SMEM) {
            g_create_error = "device has too little shared memory per block for the product kernel";
            nbs_destroy(c);
            return NBS_ECUDA;
        }
        c->prod_grid = prop.multiProcessorCount;
        smem_optin = (size_t)prop.sharedMemPerBlockOptin;
        // pipelined kernel: needs a program (Plan::cprog_ok) and room for three record buffers
        c->c_units_bytes = (uint32_t)c->plan.max_pair_units * (uint32_t)sizeof(Unit3Rec);
        c->c_rec_stride = C_ITEM_BYTES + c->c_units_bytes + (uint32_t)c->plan.max_pair_diags * (uint32_t)sizeof(Diag3Rec);
        c->c_smem = cprod_smem_bytes(c->c_rec_stride);
        c->use_c = c->plan.cprog_ok && c->c_smem <= (size_t)prop.sharedMemPerBlockOptin && c->plan.baryons.size() < 256;
        c->pipelined = c->use_c;
    }
    if (c->use_c) {
        CUC(upload(c, c->d_tabc, c->plan.tabc));
        CUC(upload(c, c->d_diagsc, c->plan.diagsc));
        CUC(upload(c, c->d_cprog, c->plan.cprog));
        CUC(upload(c, c->d_cloads, c->plan.cloads));
        std::vector<int> off, off_iso;
        std::vector<double> sg, sg_iso;
        for (size_t i = 0; i < c->plan.baryons.size(); ++i) {
            off.push_back(c->plan.slot_off[i]);
            off_iso.push_back(c->plan.slot_off[c->plan.slot_partner_iso[i]]);
        }
        for (auto& pr : c->plan.pairs3) {
            sg.push_back(1.0);
            sg_iso.push_back((double)(c->plan.slot_sign_iso[pr.slot1] * c->plan.slot_sign_iso[pr.slot2]));
        }
        CUC(upload(c, c->d_slot_off, off));
        CUC(upload(c, c->d_slot_off_iso, off_iso));
        CUC(upload(c, c->d_pair_sign, sg));
        CUC(upload(c, c->d_pair_sign_iso, sg_iso));
        CUC(build_iso_channels(c, smem_optin));
    }
    CUC(upload(c, c->d_baryon_of_slot, c->plan.baryons));
    CUC(upload(c, c->d_one_baryon, std::vector<int>(NBS_NUM_BARYONS, 0)));
    {
        std::vector<int> ids(NBS_NUM_BARYONS);
        for (int b = 0; b < NBS_NUM_BARYONS; ++b) ids[b] = b;
        CUX(cudaMemcpy(c->d_one_baryon, ids.data(), ids.size() * sizeof(int), cudaMemcpyHostToDevice));
    }
    {
        std::vector<int2> info, one;
        for (size_t i = 0; i < c->plan.baryons.size(); ++i) info.push_back(make_int2(c->plan.slot_off[i], c->plan.slot_kind[i]));
        for (int b = 0; b < NBS_NUM_BARYONS; ++b) one.push_back(make_int2(0, block_kind(b)));
        CUC(upload(c, c->d_slot_info, info));
        CUC(upload(c, c->d_gather, c->plan.gather));
        CUC(upload(c, c->d_gather_iso, c->plan.gather_iso));
        CUC(upload(c, c->d_slot_src, c->plan.slot_src));
        CUC(upload(c, c->d_one_slot_info, one));
    }
    CUC(upload(c, c->d_brec, brec));
    {
        std::vector<uint16_t> oo(3 * BLOCKS_THREADS * 16);
        blocks_out_offsets(oo.data());
        CUC(upload(c, c->d_blk_out, oo));
    }
    CUC(upload(c, c->d_bterm, bterm));
    CUC(upload(c, c->d_tw, tw));

    // workspace: per slice in flight, blocks + elementary correlators + channel correlators
    size_t nchan = c->plan.channels.size();
    size_t scratch_elems = (size_t)c->prod_grid * PROD_NBUF * c->plan.max_pair_units * 256;
    // the expanded antisymmetric blocks (Be) exist only where the one-buffer kernel runs: without a program for the
    // pipelined kernel, and for the direct shifted sum (allocated by nbs_set_direct)
    const size_t Re_res = c->use_c ? 0 : c->Re;
    size_t per_slice = (c->V * (c->R + Re_res + nchan * 256) + scratch_elems) * sizeof(double2);
    size_t free_b = 0, total_b = 0;
    CUX(cudaMemGetInfo(&free_b, &total_b));
    size_t avail = (size_t)(0.92 * (double)free_b);
    if (budget && budget < avail + c->workspace) avail = budget > c->workspace ? budget - c->workspace : 0;
    c->nslices = (T >= 2 && 2 * per_slice <= avail) ? 2 : 1;
    c->ft_rows = nchan;
    size_t chunk_elems = 0;
    if (per_slice > avail) {
        // tile-wise plan: chunks of two sink-spin planes, Ft for the channels of one sink pair, at least two chunks
        size_t maxchan = 1;
        for (auto& pr : c->plan.pairs3) maxchan = std::max<size_t>(maxchan, (size_t)pr.nchan);
        chunk_elems = c->V * (size_t)(2 * SM_PLANE);
        const size_t fixed = (c->V * maxchan * 256 + scratch_elems + 1) * sizeof(double2);
        const size_t chunk_bytes = chunk_elems * sizeof(double2);
        const size_t nfit = avail > fixed ? (avail - fixed) / chunk_bytes : 0;
        if (nfit < 2) {
            g_create_error = "neither the resident workspace (" + std::to_string(per_slice) + " bytes per time slice) nor the "
                             "tile-wise plan (" + std::to_string(fixed + 2 * chunk_bytes) + " bytes) fits (" +
                             std::to_string(avail) + " available)";
            nbs_destroy(c);
            return NBS_ENOMEM;
        }
        c->tiled = true;
        c->use_c = c->pipelined = false;
        c->nslices = 1;
        c->ft_rows = maxchan;
        c->chunks.resize(std::min<size_t>(nfit, 2 * c->plan.baryons.size()));
    }
    for (int i = 0; i < c->nslices; ++i) {
        if (!c->tiled) {
            CUC(dev_alloc(c, c->slice[i].B, c->V * c->R));
            if (!c->use_c) CUC(dev_alloc(c, c->slice[i].Be, std::max<size_t>(c->V * c->Re, 1)));
        } else {
            for (auto& ck : c->chunks) CUC(dev_alloc(c, ck.buf, chunk_elems));
        }
        CUC(dev_alloc(c, c->slice[i].Ft, c->V * c->ft_rows * 256));
        CUC(dev_alloc(c, c->slice[i].scratch, scratch_elems));
        double2* cnt = nullptr;
        CUC(dev_alloc(c, cnt, 1));
        c->slice[i].counter = (unsigned long long*)cnt;
        CUX(cudaEventCreateWithFlags(&c->slice[i].done, cudaEventDisableTiming));
    }
    CUX(cudaFuncSetAttribute(k_product_t<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PROD_SMEM));
    CUX(cudaFuncSetAttribute(k_product_t<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PROD_SMEM));
    if (c->use_c) CUX(cudaFuncSetAttribute(k_product_c<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->c_smem));
    if (c->isoch.ok) CUX(cudaFuncSetAttribute(k_product_c<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->isoch.smem));
    CUX(cudaFuncSetAttribute(k_fft_axis_r3<32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_r3_smem_bytes<32>()));
    CUX(cudaFuncSetAttribute(k_fft_axis_r3<32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_r3_smem_bytes<32>()));
    CUX(cudaFuncSetAttribute(k_fft_axis_r3<16, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_r3_smem_bytes<16>()));
    CUX(cudaFuncSetAttribute(k_fft_axis_r3<16, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_r3_smem_bytes<16>()));
    CUX(cudaFuncSetAttribute(k_blocks, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)blocks_smem_bytes(9)));
#define NBS_XY_ATTR(L_, INV_, TOUT_) \
    CUX(cudaFuncSetAttribute(k_fft_xy<L_, INV_, TOUT_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_xy_smem_bytes<L_, TOUT_>()))
    NBS_XY_ATTR(32, false, false); NBS_XY_ATTR(32, true, false); NBS_XY_ATTR(32, true, true);
    NBS_XY_ATTR(16, false, false); NBS_XY_ATTR(16, true, false); NBS_XY_ATTR(16, true, true);
#undef NBS_XY_ATTR
    *out = c;
    return NBS_OK;
#undef CUC
#undef CUX
}

int nbs_load_propagators(nbs_ctx* c, int t, const void* u, const void* d, const void* s, int memloc, void* stream) {
    if (!c) return NBS_EINVAL;
    if (c->cuda_failed) return NBS_ECUDA;
    if (t < 0 || t >= c->T || !u || !d || !s) return fail(c, NBS_EINVAL, "bad slice index or NULL propagator");
    if (memloc != NBS_MEM_DEVICE && memloc != NBS_MEM_HOST) return fail(c, NBS_EINVAL, "bad memloc");
    CU(c, cudaSetDevice(c->device));
    cudaStream_t st = (cudaStream_t)stream;
    Slice& sl = c->slice[t % c->nslices];
    const void* src[3] = {u, d, s};
    {
        int rc = slot_acquire(c, sl, st);
        if (rc) return rc;
    }
    if (memloc == NBS_MEM_DEVICE) {
        for (int f = 0; f < 3; ++f) sl.S[f] = (const double2*)src[f];
    } else {
        size_t n = c->V * 144;
        for (int f = 0; f < 3; ++f) {
            int alias = -1;
            for (int g = 0; g < f; ++g)
                if (src[g] == src[f]) alias = g;
            if (alias >= 0) { sl.S[f] = sl.S[alias]; continue; }
            if (!sl.own[f]) {
                int rc = dev_alloc(c, sl.own[f], n);
                if (rc) return rc;
            }
            CU(c, cudaMemcpyAsync(sl.own[f], src[f], n * sizeof(double2), cudaMemcpyHostToDevice, st));
            sl.S[f] = sl.own[f];
        }
    }
    sl.t = t;
    for (auto& ck : c->chunks) ck.slot = ck.pp = -1; // chunks of the previous slice are stale
    return slot_release(c, sl, st);
}

int nbs_num_slots(const nbs_ctx* c) { return c ? c->nslices : NBS_EINVAL; }

int nbs_blocks_x(nbs_ctx* c, int t, int baryon, void* out_dev, size_t out_bytes, void* stream) {
    if (!c) return NBS_EINVAL;
    if (c->cuda_failed) return NBS_ECUDA;
    if (baryon < 0 || baryon >= NBS_NUM_BARYONS || !out_dev) return fail(c, NBS_EINVAL, "bad baryon id or NULL output");
    if (t < 0 || t >= c->T) return fail(c, NBS_EINVAL, "bad slice index");
    Slice& sl = c->slice[t % c->nslices];
    if (sl.t != t) return fail(c, NBS_ESTATE, "time slice not loaded");
    if (out_bytes < c->V * BLOCK_ELEMS * sizeof(double2)) return fail(c, NBS_EINVAL, "output buffer too small");
    CU(c, cudaSetDevice(c->device));
    // the kernel writes the staged layout; convert to [site][alpha][xi1][xi2][xi3] for the caller
    cudaStream_t st = (cudaStream_t)stream;
    double2* tmp = nullptr;
    const int kind = block_kind(baryon);
    int rc = slot_acquire(c, sl, st);
    if (rc) return rc;
    // stream-ordered temporary: no device-wide synchronisation, freed when the stream has passed the kernels
    CU(c, cudaMallocAsync((void**)&tmp, c->V * (size_t)block_elems(kind) * sizeof(double2), st));
    rc = launch_blocks(c, sl, c->d_one_baryon + baryon, c->d_one_slot_info + baryon, 1, c->dq_mask_of[baryon], tmp,
                       (size_t)block_elems(kind), st);
    if (rc == NBS_OK) {
        const size_t n = c->V * (size_t)BLOCK_ELEMS;
        k_unstage<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(tmp, c->V, kind, (double2*)out_dev);
        ++c->launches;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) rc = cuda_fail(c, e, "nbs_blocks_x");
    }
    CU(c, cudaFreeAsync(tmp, st));
    if (rc) return rc;
    return slot_release(c, sl, st);
}

// ---- nbs_blocks_x without allocation (include/nbs.h, nbs_blocks_x_static) ----------------------------------------
// Staged block rows of one baryon between k_blocks and k_unstage, in the library image: every GPU that loads the
// library holds these NBS_STATIC_SCRATCH_BYTES until the process exits; all calls on a device share them.
static __device__ __align__(256) unsigned char g_static_scratch[NBS_STATIC_SCRATCH_BYTES];

namespace {
// In host code `g_static_scratch` names a host-side stand-in, not device memory: the kernels get the address that
// cudaGetSymbolAddress reports for the current device, looked up once per device and kept here.
constexpr int STATIC_SCRATCH_MAX_DEVICES = 64;
std::mutex g_static_scratch_mutex;
void* g_static_scratch_addr[STATIC_SCRATCH_MAX_DEVICES] = {};

int static_scratch_addr(nbs_ctx* c, double2** out) { // device c->device is current
    if (c->device < 0 || c->device >= STATIC_SCRATCH_MAX_DEVICES) return fail(c, NBS_EINVAL, "device ordinal beyond the static scratch table");
    std::lock_guard<std::mutex> lock(g_static_scratch_mutex);
    void*& p = g_static_scratch_addr[c->device];
    if (!p) {
        void* q = nullptr;
        CU(c, cudaGetSymbolAddress(&q, g_static_scratch));
        if (!q || (reinterpret_cast<uintptr_t>(q) & 255u)) return fail(c, NBS_ECUDA, "static scratch array has no aligned device address");
        p = q;
    }
    *out = static_cast<double2*>(p);
    return NBS_OK;
}
} // namespace

int nbs_blocks_x_static(nbs_ctx* c, int t, int baryon, void* out_dev, size_t out_bytes, void* stream) {
    if (!c) return NBS_EINVAL;
    if (c->cuda_failed) return NBS_ECUDA;
    if (baryon < 0 || baryon >= NBS_NUM_BARYONS || !out_dev) return fail(c, NBS_EINVAL, "bad baryon id or NULL output");
    if (t < 0 || t >= c->T) return fail(c, NBS_EINVAL, "bad slice index");
    Slice& sl = c->slice[t % c->nslices];
    if (sl.t != t) return fail(c, NBS_ESTATE, "time slice not loaded");
    if (out_bytes < c->V * BLOCK_ELEMS * sizeof(double2)) return fail(c, NBS_EINVAL, "output buffer too small");
    const int kind = block_kind(baryon);
    const size_t need = c->V * (size_t)block_elems(kind) * sizeof(double2);
    if (need > (size_t)NBS_STATIC_SCRATCH_BYTES)
        return fail(c, NBS_EINVAL, "nbs_blocks_x_static: the staged block rows of this baryon need " + std::to_string(need) +
                                       " bytes of scratch, the static scratch array holds " +
                                       std::to_string((size_t)NBS_STATIC_SCRATCH_BYTES) + " (NBS_STATIC_SCRATCH_BYTES); use nbs_blocks_x");
    CU(c, cudaSetDevice(c->device));
    double2* tmp = nullptr;
    int rc = static_scratch_addr(c, &tmp);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = slot_acquire(c, sl, st);
    if (rc) return rc;
    // k_blocks writes every staged entry k_unstage reads (zero pads of the compact rows included): nothing of the
    // previous call's contents survives into this call's output, and nothing has to be cleared
    rc = launch_blocks(c, sl, c->d_one_baryon + baryon, c->d_one_slot_info + baryon, 1, c->dq_mask_of[baryon], tmp,
                       (size_t)block_elems(kind), st);
    if (rc) return rc;
    const size_t n = c->V * (size_t)BLOCK_ELEMS;
    k_unstage<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(tmp, c->V, kind, (double2*)out_dev);
    ++c->launches;
    CU(c, cudaGetLastError());
    return slot_release(c, sl, st);
}

int nbs_correlator(nbs_ctx* c, int t, int ch_begin, int ch_end, void* out, size_t out_bytes, int memloc, void* stream) {
    if (!c) return NBS_EINVAL;
    if (c->cuda_failed) return NBS_ECUDA;
    const int nch = (int)c->plan.channels.size();
    if (t < 0 || t >= c->T) return fail(c, NBS_EINVAL, "bad slice index");
    if (ch_begin < 0 || ch_end > nch || ch_begin >= ch_end || !out) return fail(c, NBS_EINVAL, "bad channel range or NULL output");
    if (memloc != NBS_MEM_DEVICE && memloc != NBS_MEM_HOST) return fail(c, NBS_EINVAL, "bad memloc");
    const size_t nout = (size_t)(ch_end - ch_begin);
    const size_t need = nout * 256 * c->V * sizeof(double2);
    if (out_bytes < need) return fail(c, NBS_EINVAL, "output buffer too small");
    Slice& sl = c->slice[t % c->nslices];
    if (sl.t != t) return fail(c, NBS_ESTATE, "time slice not loaded");
    CU(c, cudaSetDevice(c->device));
    cudaStream_t st = (cudaStream_t)stream;
    // host output: the result is staged in a block buffer (free again after the product) and copied back; the
    // range must fit BEFORE anything is enqueued
    if (c->tiled) {
        int rc0 = slot_acquire(c, sl, st);
        if (rc0) return rc0;
        rc0 = correlator_tiled(c, sl, ch_begin, ch_end, out, memloc, st);
        if (rc0) return rc0;
        return slot_release(c, sl, st);
    }
    double2* dst = (double2*)out;
    if (memloc == NBS_MEM_HOST) {
        if (need <= c->V * c->R * sizeof(double2)) dst = sl.B;
        else if (sl.Be && need <= c->V * c->Re * sizeof(double2)) dst = sl.Be;
        else return fail(c, NBS_ENOMEM, "channel range too large for the device staging of a host output; use a smaller range");
    }
    {
        int rc0 = slot_acquire(c, sl, st);
        if (rc0) return rc0;
    }

    // isospin-limit fast path: the caller passed the same array for u and d
    const bool iso = sl.S[0] == sl.S[1] && c->plan.n_slots_iso < (int)c->plan.baryons.size();
    // (i) normal baryon blocks, then forward FFT in place
    int rc;
    {
        StageTimer tm(c, NBS_STAGE_BLOCKS, st);
        rc = launch_blocks(c, sl, c->d_baryon_of_slot, c->d_slot_info, iso ? c->plan.n_slots_iso : (int)c->plan.baryons.size(),
                           iso ? c->dq_mask_iso : c->dq_mask, sl.B, c->R, st);
        if (rc) return rc;
    }
    {
        StageTimer tm(c, NBS_STAGE_FFT_FWD, st);
        if (!c->direct) {
            rc = fft3d(c, sl.B, c->R, false, st, nullptr, iso ? (size_t)c->plan.row_elems_iso : 0);
            if (rc) return rc;
        }
        const bool pipelined = c->pipelined && !c->direct;
        if (c->Re && !pipelined) { // antisymmetric blocks: mirror halves restored for the gathers of the one-buffer kernel
            k_expand<<<(unsigned)c->V, 256, 0, st>>>(sl.B, c->R, iso ? c->d_gather_iso : c->d_gather, (int)c->Re, sl.Be);
            CU(c, cudaGetLastError());
            ++c->launches;
        }
    }
    // (ii)+(iii) effective blocks and their products -> elementary correlators -> channels
    {
        StageTimer tm(c, NBS_STAGE_PRODUCT, st);
        CU(c, cudaMemsetAsync(sl.counter, 0, sizeof(unsigned long long), st));
        const bool pipelined = c->pipelined && !c->direct;
        ProdArgs pa;
        pa.Bc = sl.B; pa.Rc = c->R; pa.Be = sl.Be; pa.Re = c->Re; pa.L = c->L;
        pa.slot_src = reinterpret_cast<const int2*>(c->d_slot_src);
        pa.chain_full_n = c->plan.chain_full_n; pa.chain_half_n = c->plan.chain_half_n;
        pa.ntasks = c->direct ? (long long)c->V : c->ntasks; // direct: one task per displacement r
        pa.direct = c->direct ? 1 : 0;
        pa.qorder = c->d_qorder;
        pa.pairs = c->d_pairs3; pa.units = c->d_units3; pa.diags = c->d_diags3;
        pa.tab = reinterpret_cast<const uint2*>(c->d_tab3);
        pa.pair_chans = c->d_pair_chans; pa.chain = c->d_chain;
        pa.scratch = sl.scratch; pa.max_pair_units = c->plan.max_pair_units;
        pa.Ft = sl.Ft; pa.ch_begin = ch_begin; pa.nch_out = (int)nout;
        pa.counter = sl.counter;
        unsigned grid = (unsigned)std::min<long long>(c->prod_grid, pa.ntasks);
        pa.c1 = pa.c2 = nullptr; pa.tile_i = pa.tile_j = 0; pa.chain_base = 0;
        if (pipelined) {
            CProdArgs ca;
            ca.base = pa;
            ca.B = sl.B; ca.R = c->R;
            ca.slot_off = iso ? c->d_slot_off_iso : c->d_slot_off;
            ca.pair_sign = iso ? c->d_pair_sign_iso : c->d_pair_sign;
            ca.ntasks = c->ntasks_half; ca.qhalf = c->d_qorder_half;
            ca.prog = c->d_cprog; ca.nitems = (int)c->plan.cprog.size(); ca.loads = c->d_cloads;
            ca.units = c->d_units3; ca.diags = c->d_diagsc; ca.tab = c->d_tabc;
            ca.rec_stride = c->c_rec_stride; ca.units_bytes = c->c_units_bytes;
            size_t smem = c->c_smem;
            const bool alias = iso && c->isoch.ok && c->iso_relations;
            if (alias) { // channels that are u <-> d images are written from their originals
                const nbs_ctx::IsoChannels& ic = c->isoch;
                ca.base.pairs = ic.d_pairs3; ca.base.pair_chans = ic.d_pair_chans; ca.base.max_pair_units = ic.plan.max_pair_units;
                ca.slot_off = ic.d_slot_off; ca.pair_sign = ic.d_pair_sign;
                ca.prog = ic.d_cprog; ca.nitems = (int)ic.plan.cprog.size(); ca.loads = ic.d_cloads;
                ca.units = ic.d_units3; ca.diags = ic.d_diagsc; ca.tab = ic.d_tabc;
                ca.rec_stride = ic.rec_stride; ca.units_bytes = ic.units_bytes;
                smem = ic.smem;
            }
            grid = (unsigned)std::min<long long>(c->prod_grid, ca.ntasks);
            if (alias) k_product_c<true><<<grid, C_THREADS, smem, st>>>(ca);
            else k_product_c<false><<<grid, C_THREADS, smem, st>>>(ca);
        } else
        k_product_t<false><<<grid, PROD_THREADS, PROD_SMEM, st>>>(pa);
        CU(c, cudaGetLastError());
        ++c->launches;
    }
    // inverse FFT and final layout F[ch][a1 a2 a3 a4][r]
    const bool fused = fft_fused(c) && !c->direct;
    if (!c->direct) {
        StageTimer tm(c, NBS_STAGE_FFT_INV, st);
        rc = fft3d(c, sl.Ft, nout * 256, true, st, fused ? dst : nullptr);
        if (rc) return rc;
    }
    if (!fused) {
        StageTimer tm(c, NBS_STAGE_OUTPUT, st);
        dim3 tg((unsigned)((c->V + 31) / 32), (unsigned)((nout * 256 + 31) / 32));
        k_transpose_out<<<tg, 256, 0, st>>>(sl.Ft, c->V, nout * 256, nout * 256, dst);
        CU(c, cudaGetLastError());
        ++c->launches;
    }
    if (memloc == NBS_MEM_HOST) CU(c, cudaMemcpyAsync(out, dst, need, cudaMemcpyDeviceToHost, st));
    return slot_release(c, sl, st);
}

// the expanded antisymmetric blocks of the one-buffer kernel exist only once somebody asks for that kernel
static int ensure_expanded(nbs_ctx* c) {
    if (!c->Re || c->tiled) return NBS_OK;
    for (int i = 0; i < c->nslices; ++i)
        if (!c->slice[i].Be) {
            CU(c, cudaSetDevice(c->device));
            int rc = dev_alloc(c, c->slice[i].Be, c->V * c->Re);
            if (rc) return rc;
        }
    return NBS_OK;
}

int nbs_set_direct(nbs_ctx* c, int enable) {
    if (!c) return NBS_EINVAL;
    if (enable && c->L > 8) return fail(c, NBS_EINVAL, "the direct shifted sum is O(V^2): allowed for L <= 8 only");
    if (enable && c->tiled) return fail(c, NBS_EINVAL, "the direct shifted sum is not available with the tile-wise plan");
    if (enable) { // the direct sum runs the one-buffer kernel on expanded x-space blocks
        int rc = ensure_expanded(c);
        if (rc) return rc;
    }
    c->direct = enable != 0;
    return NBS_OK;
}

int nbs_set_pipelined(nbs_ctx* c, int enable) {
    if (!c) return NBS_EINVAL;
    if (enable < 0) return c->pipelined ? 1 : 0; // query
    if (enable && !c->use_c) return fail(c, NBS_EINVAL, "the pipelined product kernel is not available for this plan (fewer than 3 sink-pair items per momentum pair, tile-wise plan, or too many unit records for shared memory)");
    if (!enable) {
        int rc = ensure_expanded(c);
        if (rc) return rc;
    }
    c->pipelined = enable != 0;
    return NBS_OK;
}

int nbs_set_timing(nbs_ctx* c, int enable) {
    if (!c) return NBS_EINVAL;
    c->timing = enable != 0;
    return NBS_OK;
}

int nbs_stage_times(nbs_ctx* c, double* ms, long long* calls, int reset) {
    if (!c) return NBS_EINVAL;
    if (c->cuda_failed) return NBS_ECUDA;
    for (auto& p : c->pending) {
        CU(c, cudaEventSynchronize(p.b));
        float t = 0.f;
        CU(c, cudaEventElapsedTime(&t, p.a, p.b));
        c->stage_ms[p.stage] += t;
        c->stage_calls[p.stage] += 1;
        c->event_pool.push_back(p.a);
        c->event_pool.push_back(p.b);
    }
    c->pending.clear();
#ifdef NBS_PROF
    {
        unsigned long long pf[PF_N] = {}, zero[PF_N] = {};
        cudaMemcpyFromSymbol(pf, g_cprof, sizeof(pf));
        cudaMemcpyToSymbol(g_cprof, zero, sizeof(zero));
        static const char* names[PF_N] = {"total", "units", "wait_empty", "wait_rec", "wait_slot", "release", "multi_term_diagrams"};
        if (pf[PF_TOTAL]) {
            fprintf(stderr, "[NBS_PROF] compute-warp cycles:");
            for (int i = 0; i < PF_N; ++i) fprintf(stderr, " %s %.2f%%", names[i], 100.0 * (double)pf[i] / (double)pf[PF_TOTAL]);
            fprintf(stderr, "\n");
        }
    }
#endif
    for (int i = 0; i < NBS_NUM_STAGES; ++i) {
        if (ms) ms[i] = c->stage_ms[i];
        if (calls) calls[i] = c->stage_calls[i];
        if (reset) { c->stage_ms[i] = 0; c->stage_calls[i] = 0; }
    }
    return NBS_OK;
}

void nbs_destroy(nbs_ctx* c) {
    if (!c) return;
    if (cudaSetDevice(c->device) == cudaSuccess) {
        cudaDeviceSynchronize();
        for (void* p : c->allocs) cudaFree(p);
        for (auto& p : c->pending) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
        for (cudaEvent_t e : c->event_pool) cudaEventDestroy(e);
        for (auto& sl : c->slice) if (sl.done) cudaEventDestroy(sl.done);
    }
    delete c;
}

const char* nbs_last_error(const nbs_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }
size_t nbs_workspace_bytes(const nbs_ctx* c) { return c ? c->workspace : 0; }
int nbs_num_channels(const nbs_ctx* c) { return c ? (int)c->plan.channels.size() : NBS_EINVAL; }
int nbs_channel_info(const nbs_ctx* c, int i, nbs_channel* out) {
    if (!c || !out || i < 0 || i >= (int)c->plan.channels.size()) return NBS_EINVAL;
    *out = c->plan.channels[i];
    return NBS_OK;
}

int nbs_model_flops(const nbs_ctx* c, double* blocks, double* fft, double* product) {
    if (!c) return NBS_EINVAL;
    // complex multiply-add = 8 flops.  Blocks: per distinct (f0 f1 f2) tensor 432*8 + 6912*3 cMAC.
    std::vector<int> seen;
    for (int b : c->plan.baryons)
        for (auto& t : block_terms(b)) {
            int key = (t.f0 * 3 + t.f1) * 3 + t.f2;
            bool have = false;
            for (int k : seen) have = have || (k == key);
            if (!have) seen.push_back(key);
        }
    if (blocks) *blocks = 8.0 * seen.size() * (432.0 * 8 + 6912.0 * 3);
    double lg = std::log2((double)c->V);
    if (fft) *fft = 5.0 * lg * ((double)c->R + 256.0 * c->plan.channels.size());
    if (product) *product = 8.0 * 256.0 * c->plan.sumK_std;
    return NBS_OK;
}

int nbs_exec_flops(const nbs_ctx* c, double* product_executed) {
    if (!c) return NBS_EINVAL;
    // pairs of identical sink baryons are computed for the momenta q <= -q only
    const double self_frac = 0.5 * (double)(c->V + c->nselfconj) / (double)c->V;
    if (product_executed) *product_executed = 8.0 * 256.0 * (c->plan.sumK_exec + self_frac * c->plan.sumK_exec_self);
    return NBS_OK;
}

int nbs_fft3d(nbs_ctx* c, void* data_dev, size_t R, int inverse, void* stream) {
    if (!c) return NBS_EINVAL;
    if (c->cuda_failed) return NBS_ECUDA;
    if (!data_dev || R == 0) return fail(c, NBS_EINVAL, "NULL data or R == 0");
    if (reinterpret_cast<uintptr_t>(data_dev) & 15u) return fail(c, NBS_EINVAL, "data must be 16-byte aligned");
    CU(c, cudaSetDevice(c->device));
    return fft3d(c, (double2*)data_dev, R, inverse != 0, (cudaStream_t)stream);
}

int nbs_probe_kstep(nbs_ctx* c, int cls, int warps, int nsteps, int reps, double* cycles_per_kstep, double* cycles_max) {
    if (!c) return NBS_EINVAL;
    if (c->cuda_failed) return NBS_ECUDA;
    if ((cls != 0 && cls != 2) || warps < 1 || warps > PROBE_KSTEP_THREADS / 32 || nsteps < 1 || nsteps > PROBE_KSTEP_MAX_STEPS || reps < 1)
        return fail(c, NBS_EINVAL, "nbs_probe_kstep: cls 0 or 2, 1 <= warps <= 12, 1 <= nsteps <= 48, reps >= 1");
    CU(c, cudaSetDevice(c->device));
    // packed gather words whose four consecutive k fall into four different bank groups modulo 4 (what the real
    // tables guarantee): offset = 16 * (4 * random + k mod 4); k = (word / 4) mod 4, or (word / 16) mod 4 in the
    // A table of the 64 x 4 class ([k][cX & 3][g])
    std::vector<uint32_t> tab(PROBE_KSTEP_TAB_WORDS);
    uint32_t rng = 12345u;
    auto next = [&] { rng = rng * 1664525u + 1013904223u; return (rng >> 10) % 200u; };
    for (size_t i = 0; i < tab.size(); ++i) {
        const uint32_t k = (cls >= 2 && i < 65536) ? (uint32_t)((i / 16) % 4) : (uint32_t)((i / 4) % 4);
        tab[i] = ((next() * 4 + k) * 16u) | (((next() * 4 + k) * 16u) << 16);
    }
    const int grid = c->prod_grid, nw = PROBE_KSTEP_THREADS / 32;
    uint32_t* d_tab = nullptr; double2* d_out = nullptr; long long* d_cyc = nullptr;
    CU(c, cudaMalloc((void**)&d_tab, tab.size() * sizeof(uint32_t)));
    CU(c, cudaMalloc((void**)&d_out, (size_t)grid * nw * 256 * sizeof(double2)));
    CU(c, cudaMalloc((void**)&d_cyc, (size_t)grid * nw * sizeof(long long)));
    cudaError_t e = cudaMemcpy(d_tab, tab.data(), tab.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(d_cyc, 0, (size_t)grid * nw * sizeof(long long));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_probe_kstep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C_BLOCKS_BYTES);
    std::vector<long long> cyc((size_t)grid * nw, 0);
    if (e == cudaSuccess) {
        k_probe_kstep<<<grid, PROBE_KSTEP_THREADS, C_BLOCKS_BYTES>>>(d_tab, cls, nsteps, reps, warps, d_out, d_cyc);
        e = cudaDeviceSynchronize();
    }
    if (e == cudaSuccess) e = cudaMemcpy(cyc.data(), d_cyc, cyc.size() * sizeof(long long), cudaMemcpyDeviceToHost);
    cudaFree(d_tab); cudaFree(d_out); cudaFree(d_cyc);
    if (e != cudaSuccess) return cuda_fail(c, e, "nbs_probe_kstep");
    ++c->launches;
    double sum = 0.0, mx = 0.0;
    for (int b = 0; b < grid; ++b)
        for (int w = 0; w < warps; ++w) {
            const double v = (double)cyc[(size_t)b * nw + w] / ((double)reps * nsteps);
            sum += v; mx = std::max(mx, v);
        }
    if (cycles_per_kstep) *cycles_per_kstep = sum / ((double)grid * warps);
    if (cycles_max) *cycles_max = mx;
    return NBS_OK;
}

long long nbs_kernel_launches(const nbs_ctx* c) { return c ? c->launches : 0; }

int nbs_pair_order(const nbs_ctx* c, int* ch_begin, int* ch_end, int cap) {
    if (!c) return NBS_EINVAL;
    const Plan& P = c->plan;
    for (int ci = 0; ci < P.chain_full_n; ++ci) {
        const Pair3Rec& pr = P.pairs3[P.chain[ci].pair];
        int lo = 1 << 30, hi = -1;
        for (int k = 0; k < pr.nchan; ++k) {
            const int ch = P.pair_chans[pr.chan_begin + k].ch;
            lo = std::min(lo, ch); hi = std::max(hi, ch + 1);
        }
        if (ci < cap) {
            if (ch_begin) ch_begin[ci] = lo;
            if (ch_end) ch_end[ci] = hi;
        }
    }
    return P.chain_full_n;
}

int nbs_tiled_info(const nbs_ctx* c, int* chunk_slots, long long* chunk_builds) {
    if (!c) return NBS_EINVAL;
    if (chunk_slots) *chunk_slots = (int)c->chunks.size();
    if (chunk_builds) *chunk_builds = c->chunk_builds;
    return c->tiled ? 1 : 0;
}

int nbs_probe_fp64(nbs_ctx* c, int mode, int iters, double* tflops, double* ms_out) {
    if (!c) return NBS_EINVAL;
    if (c->cuda_failed) return NBS_ECUDA;
    if (mode < 0 || mode > 8 || iters < 1) return fail(c, NBS_EINVAL, "nbs_probe_fp64: mode in [0, 8], iters >= 1");
    CU(c, cudaSetDevice(c->device));
    cudaEvent_t a = nullptr, b = nullptr;
    CU(c, cudaEventCreate(&a));
    CU(c, cudaEventCreate(&b));
    double* sink = reinterpret_cast<double*>(c->slice[0].scratch); // never written (the guard in the kernel is false)
    const unsigned grid = (unsigned)c->prod_grid;
    auto launch = [&](int n) {
        switch (mode) {
        case 0: k_probe_fp64<0><<<grid, PROBE_THREADS>>>(n, 1e-9, sink); break;
        case 1: k_probe_fp64<1><<<grid, PROBE_THREADS>>>(n, 1e-9, sink); break;
        case 2: k_probe_fp64<2><<<grid, PROBE_THREADS>>>(n, 1e-9, sink); break;
        case 3: k_probe_fp64<3><<<grid, PROBE_THREADS>>>(n, 1e-9, sink); break;
        case 4: k_probe_fp64<4><<<grid, PROBE_THREADS>>>(n, 1e-9, sink); break;
        case 5: k_probe_fp64<5><<<grid, PROBE_THREADS>>>(n, 1e-9, sink); break;
        case 6: k_probe_fp64<6><<<grid, PROBE_THREADS>>>(n, 1e-9, sink); break;
        case 7: k_probe_fp64<7><<<grid, PROBE_THREADS>>>(n, 1e-9, sink); break;
        default: k_probe_fp64<8><<<grid, PROBE_THREADS>>>(n, 1e-9, sink); break;
        }
    };
    launch(iters / 8 + 1); // warm-up
    CU(c, cudaEventRecord(a, 0));
    launch(iters);
    CU(c, cudaEventRecord(b, 0));
    cudaError_t e = cudaEventSynchronize(b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    if (e != cudaSuccess) return cuda_fail(c, e, "nbs_probe_fp64");
    c->launches += 2;
    // per warp instruction: DMMA.8x8x4 = 8*8*4 FMA = 512 flop, DFMA = 32 lanes x 2, DADD = 32 lanes x 1
    const double per_iter = 512.0 * probe_dmma(mode) + 64.0 * probe_dfma(mode) + 32.0 * probe_dadd(mode);
    const double warps = (double)grid * (PROBE_THREADS / 32);
    if (tflops) *tflops = per_iter * warps * (double)iters / ((double)ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = (double)ms;
    return NBS_OK;
}

} // extern "C"
