/*
 * nbs.h -- C ABI of the B200-native hot path of the HAL QCD effective baryon block algorithm
 * (H. Nemura, arXiv:1604.07983; citations are PAPER.md:<line>, section / equation).
 *
 * What the library computes (eq. 2.1; eq. 2.4; eq. 2.6):
 * for one time slice t and each requested channel <B1 B2 | B3 B4>
 *
 *   F[ch][a1][a2][a3][a4][r] = sum_X  sum_P sigma_P [B1_a1](X+r; xi'_P1 xi'_P2 xi'_P3) [B2_a2](X; xi'_P4 xi'_P5 xi'_P6)
 *                               x eps eps (C g5)(C g5) delta delta                           (eq. 2.4)
 *
 * from the u, d, s wall-source quark propagators on that slice, via (i) normal baryon blocks
 * (eq. 2.5 / 4.1), FFT, (ii)+(iii) effective blocks and their product (eqs. 4.2, 4.3), inverse
 * FFT (eq. 2.6).  Everything runs in hand-written sm_100a CUDA kernels in complex128; there is no
 * CPU fallback: every entry point fails with NBS_ECUDA if no CUDA device is usable.
 *
 * Conventions (readings A1-A17):
 *   xi = colour + 3*spin (12 values);  site index x + L*(y + L*z);  periodic space;
 *   propagator S_f[site][sink xi][source xi'] complex128 (re, im interleaved), row-major 12x12;
 *   C gamma_5 = [[0,1,0,0],[-1,0,0,0],[0,0,0,1],[0,0,-1,0]];
 *   r = position of B1 minus position of B2;  spin index ((a1*4+a2)*4+a3)*4+a4.
 *
 * Threading: a context is not thread-safe; different contexts are independent.
 * Errors: every function returns 0 (NBS_OK) or a negative NBS_E* code; nothing throws across the
 * ABI; nbs_last_error() gives a human-readable message for the last failure on a context.
 */
#ifndef NBS_H_
#define NBS_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nbs_ctx nbs_ctx;

/* Interpolating fields of eqs. 2.2-2.3. */
enum {
    NBS_P = 0,       /* p       =  eps (u Cg5 d) u */
    NBS_N = 1,       /* n       = -eps (u Cg5 d) d */
    NBS_LAMBDA = 2,  /* Lambda  = (X_u + X_d - 2 X_s)/sqrt 6 */
    NBS_SIGMA_P = 3, /* Sigma+  = -eps (u Cg5 s) u */
    NBS_SIGMA_0 = 4, /* Sigma0  = (X_u - X_d)/sqrt 2 */
    NBS_SIGMA_M = 5, /* Sigma-  = -eps (d Cg5 s) d */
    NBS_XI_0 = 6,    /* Xi0     =  eps (u Cg5 s) s */
    NBS_XI_M = 7,    /* Xi-     = -eps (d Cg5 s) s */
    NBS_XU = 8,      /* X_u     =  eps (d Cg5 s) u   (eq. 2.3; e.g. <p Lambda pbar Xubar>, eq. 2.7) */
    NBS_XD = 9,      /* X_d     =  eps (s Cg5 u) d */
    NBS_XS = 10,     /* X_s     =  eps (u Cg5 d) s */
    NBS_NUM_BARYONS = 11
};

/* One channel <B1 B2 | B3 B4>: sink baryons b1 (at X+r), b2 (at X); source baryons b3, b4. */
typedef struct {
    int b1, b2, b3, b4;
} nbs_channel;

enum {
    NBS_OK = 0,
    NBS_EINVAL = -1,  /* bad argument: L, T, baryon id, channel violating flavour conservation, range */
    NBS_ENOMEM = -2,  /* workspace does not fit in device memory / the given budget */
    NBS_ESTATE = -3,  /* call order: slice t not loaded, context destroyed, ... */
    NBS_ECUDA = -4    /* CUDA runtime error (sticky for the context; see nbs_last_error) */
};

enum {
    NBS_MEM_DEVICE = 0, /* pointer is device memory on the context's device */
    NBS_MEM_HOST = 1    /* pointer is host memory (pinned for asynchronous copies) */
};

/*
 * nbs_create -- build the diagram tables (the paper's CPU "diagramatical classification", SoA
 * tables copied to the device before the kernels) and allocate the workspace.
 *   out       : receives the context (library-owned; free with nbs_destroy).
 *   L, T      : spatial extent: 2 <= L <= 64, or L = 3 * 2^k <= 96 (in-register radix-2 FFT for powers of two up to
 *               32, the same behind a radix-3 stage for 6, 12, 24, 48, 96, an O(L^2) transform per axis otherwise),
 *               and number of time slices (labels only: slices are independent).  With the 52 channels the
 *               resident plan needs 1.4 MB of workspace per site (46 GB at 32^3); larger lattices take the tile-wise
 *               plan (nbs_tiled_info), which needs about 2 x 55.7 KB per site plus the channels of one sink pair.
 *   ch, nch   : channel list (host memory, copied).  ch == NULL selects the standard 52 channels
 *               "from NN to Xi-Xi" in the order of DESIGN.md reading A10.
 *   device    : CUDA device ordinal.
 *   workspace_budget_bytes : upper bound for library-owned device memory (0 = no bound).  Two workspaces (two time
 *               slices in flight) if they fit, else one, else the tile-wise plan, else NBS_ENOMEM.
 * Errors: NBS_EINVAL (bad L/T/id, or a channel whose sink and source flavour content differ for
 * every elementary source term: F would vanish identically), NBS_ENOMEM, NBS_ECUDA.
 */
int nbs_create(nbs_ctx** out, int L, int T, const nbs_channel* ch, int nch, int device,
               size_t workspace_budget_bytes);

/*
 * nbs_load_propagators -- hand the u, d, s propagators of time slice t to the library
 * ("Assuming that the quark propagators are already solved").
 *   u, d, s : each [L^3][12][12] complex128 (layout above).  Pointer equality (d == u, s == u)
 *             is allowed and means the same array; d == u additionally selects the isospin-limit fast path
 *             (PAPER.md:102): the n, Sigma-, Xi- blocks are derived from p, Sigma+, Xi0 instead of being built
 *             and Fourier transformed (same results up to rounding).
 *   memloc  : NBS_MEM_DEVICE -> borrowed, must stay valid until the matching nbs_correlator(t)
 *             has completed on its stream;  NBS_MEM_HOST -> copied asynchronously on `stream`
 *             into library-owned device memory (the caller may reuse the host buffer after the
 *             stream has passed this point).
 *   stream  : a cudaStream_t (NULL = default stream).
 * Only one slice is held at a time per slot; the library keeps 2 slots (t % 2) so that two
 * slices can be in flight on two streams (cudaStream overlap).
 */
int nbs_load_propagators(nbs_ctx* ctx, int t, const void* u, const void* d, const void* s, int memloc,
                         void* stream);

/*
 * nbs_correlator -- the hot path for slice t, channels [ch_begin, ch_end):
 *   (i)  normal baryon blocks, eq. 4.1, forward FFT,
 *   (ii) effective blocks, eq. 4.2, fused with
 *   (iii) their product summed over the shared index and the diagrams, eq. 4.3,
 *   inverse FFT, eq. 2.6.
 * Writes F[ch - ch_begin][a1][a2][a3][a4][r] (complex128, r fastest) to `out`.
 *   out, out_bytes, memloc : caller-owned buffer of at least (ch_end-ch_begin)*256*L^3*16 bytes;
 *             NBS_MEM_DEVICE (written by the kernels) or NBS_MEM_HOST (device result copied back
 *             asynchronously on `stream`).
 * Asynchronous on `stream`: synchronise the stream before reading `out`.
 * Errors: NBS_ESTATE (slice t not loaded), NBS_EINVAL (range / size), NBS_ECUDA.
 */
int nbs_correlator(nbs_ctx* ctx, int t, int ch_begin, int ch_end, void* out, size_t out_bytes, int memloc,
                   void* stream);

/* nbs_destroy -- synchronise the device, free tables and workspace.  NULL is a no-op. */
void nbs_destroy(nbs_ctx* ctx);

/*
 * nbs_num_slots -- number of workspace slots (time slices that can be in flight at once): 2 when two
 * workspaces fit the budget / the free device memory and T >= 2, else 1.  Slice t uses slot t % nbs_num_slots.
 * Sharing a slot is safe: every call that touches a slot on another stream than the previous call on that slot
 * first makes its stream wait (cudaStreamWaitEvent) for that call, so slices that share a slot serialise; a
 * caller that wants overlap uses one stream per slot.
 */
int nbs_num_slots(const nbs_ctx* ctx);

/*
 * nbs_tiled_info -- which plan nbs_create chose.  Returns 0 for the resident plan (the momentum-space normal blocks
 * of a whole time slice live in device memory: every lattice up to 32^3 with the 52 channels on a B200) and 1 for
 * the tile-wise plan (BASELINE.json configs[4], 96^3: "blocks must be contracted tile-wise"), taken when the
 * resident workspace does not fit workspace_budget_bytes / the free device memory.  Tile-wise, the momentum-space
 * blocks exist only as chunks of two sink-spin planes of one baryon (49 GB at 96^3), built on demand and cached in
 * *chunk_slots buffers; nbs_correlator then runs sink pair by sink pair and plane pair by plane pair, and a channel
 * range should cover whole sink pairs (consecutive channels of the standard list) to avoid recomputation.  Results
 * are the same as with the resident plan.  *chunk_builds counts the chunks built so far.  Either pointer may be NULL.
 */
int nbs_tiled_info(const nbs_ctx* ctx, int* chunk_slots, long long* chunk_builds);

/*
 * nbs_pair_order -- the sink pairs (B1 B2) of the channel list in the order in which the library walks them
 * (consecutive pairs share a baryon block), each as the smallest channel range [ch_begin[i], ch_end[i]) that holds
 * its channels (in the standard 52-channel list the channels of a sink pair are consecutive).  With the tile-wise
 * plan, calling nbs_correlator once per range in this order builds the fewest chunks.  Returns the number of sink
 * pairs; writes at most `cap` entries; either array may be NULL.
 */
int nbs_pair_order(const nbs_ctx* ctx, int* ch_begin, int* ch_end, int cap);

/* Helpers. */
const char* nbs_last_error(const nbs_ctx* ctx); /* never NULL; ctx == NULL -> last nbs_create error */
size_t nbs_workspace_bytes(const nbs_ctx* ctx); /* library-owned device bytes */
int nbs_num_channels(const nbs_ctx* ctx);
int nbs_channel_info(const nbs_ctx* ctx, int i, nbs_channel* out);

/*
 * Table statistics of the host generator (row a0 of DESIGN.md; pins: 52 channels, 3456 literal
 * and 370 = 1+9+144+144+36+36 effective terms for <p Lambda pbar Xubar>).
 * These run on the host only (no CUDA call) so they work on a machine without a GPU.
 *   nbs_std_channels : writes the standard 52 channels to `out` (capacity `cap`), returns 52.
 *   nbs_diagram_stats: for one channel, returns the number of diagrams (coset representatives
 *             summed over elementary source terms) and writes up to `cap` shared-index sizes K_d
 *             to `K` (in enumeration order: source terms major, permutations lexicographic) and
 *             signs sigma_P to `sign`; *literal_terms receives diagrams * (N_c! N_alpha)^2.
 *             Returns NBS_EINVAL for an invalid channel.
 */
int nbs_std_channels(nbs_channel* out, int cap);
/*   nbs_plan_selfcheck: host-only bounds check of the tables the kernels index with (gather offsets inside the staged
 *             blocks, table extents including the software pipeline's look-ahead, unit / diagram / chain / channel record
 *             ranges, expansion maps); ch == NULL checks the standard 52 channels.  If the list holds u <-> d images
 *             (nbs_iso_relations), the reduced plan of the isospin limit is built and checked the same way (check numbers
 *             minus 1000), together with the mirror relation of its conjugate sink pairs (an involution inside the pair,
 *             signs +-1: -1151 ... -1155).  Returns 0 or a negative check number. */
int nbs_plan_selfcheck(const nbs_channel* ch, int nch);
int nbs_diagram_stats(const nbs_channel* ch, int* K, int* sign, int cap, long long* literal_terms);

/*
 * Stage-level entry points (used by the parity tests and by bench.py's per-stage timing).
 *   nbs_blocks_x : eq. 4.1 only: writes the x-space normal block of baryon `baryon` for the
 *             loaded slice t to device buffer out[site][alpha][xi1][xi2][xi3] (complex128).
 *   nbs_model_flops : the algorithmic flop count per lattice site for the context's channel list
 *             (complex multiply-add = 8 flops): blocks, fft (forward+inverse), product
 *             (256 * sum_d K_d over the channels' diagrams), as doubles.
 */
int nbs_blocks_x(nbs_ctx* ctx, int t, int baryon, void* out_dev, size_t out_bytes, void* stream);

/*
 * nbs_blocks_x_static -- nbs_blocks_x (eq. 4.1) for callers that must not allocate device memory
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same arguments, same
 * kernels, same result bit for bit; the only difference is where the staged block rows live between the block kernel
 * and the layout kernel: nbs_blocks_x takes them from the stream-ordered allocator (cudaMallocAsync / cudaFreeAsync),
 * this entry point uses a scratch array that is part of the library image (`static __device__`,
 * NBS_STATIC_SCRATCH_BYTES, resident on every GPU that loads the library until the process exits).  It calls no
 * cudaMalloc, cudaFree or allocating library routine; the first call on a device looks the array's device address up
 * once (cudaGetSymbolAddress, no allocation).
 *   Limit: L^3 * E * 16 <= NBS_STATIC_SCRATCH_BYTES (32 MiB) with E = 3472 staged entries per site for p, n, Sigma+-,
 *   Xi0- (antisymmetric blocks, compact rows) and 6960 for the others: L <= 8 resp. L <= 6.  Beyond it: NBS_EINVAL,
 *   with the bytes needed and the maximum in nbs_last_error; nothing is launched.
 *   Sharing: all calls on a device, from every context and stream, use the SAME array.  Calls ordered on one stream
 *   are safe; calls that may overlap on the GPU (different streams without an event between them, different host
 *   threads) race on it -- the caller serialises them.  Nothing in the array has to start at zero: the block kernel
 *   writes every staged entry the layout kernel reads, so the previous call's contents are never seen.
 * Errors as nbs_blocks_x, plus the limit above.
 */
#define NBS_STATIC_SCRATCH_BYTES (32u << 20)
int nbs_blocks_x_static(nbs_ctx* ctx, int t, int baryon, void* out_dev, size_t out_bytes, void* stream);
int nbs_model_flops(const nbs_ctx* ctx, double* blocks, double* fft, double* product);

/*
 *   nbs_exec_flops : flops per site the product kernels actually execute (8 * 256 * sum of K_d over
 *             the DISTINCT elementary correlators: source Lambda / Sigma0 terms shared between
 *             channels of one sink pair are evaluated once).  <= the `product` model count.
 *   nbs_fft3d : rows a2 / a5 alone (eq. 2.6): in-place 3-D transform of a device
 *             array data[site][R] complex128 (16-byte aligned: the x-y pass uses 16-byte asynchronous copies), every
 *             one of the R components independently.
 *             inverse == 0: sum_x f(x) exp(-i q.x);  inverse != 0: L^-3 sum_q f(q) exp(+i q.r).
 *   nbs_kernel_launches : number of CUDA kernels this context has launched so far (bench.py's
 *             `gpu_launches`).
 */
/*
 * Per-stage device timing (bench.py's roofline figures).  When enabled, nbs_correlator brackets
 * each stage with a pair of CUDA events recorded on the stream the kernels are launched on;
 * nbs_stage_times synchronises those events, adds their elapsed times to per-stage totals, writes
 * total milliseconds and number of timed stage executions for the NBS_NUM_STAGES stages
 * (either pointer may be NULL), and, if reset != 0, clears the totals.
 */
enum {
    NBS_STAGE_BLOCKS = 0,   /* (i) normal baryon blocks, eq. 4.1 */
    NBS_STAGE_FFT_FWD = 1,  /* forward FFT of the block components (+ expansion of the antisymmetric blocks) */
    NBS_STAGE_PRODUCT = 2,  /* (ii)+(iii) effective blocks and their product, eqs. 4.2-4.3 */
    NBS_STAGE_FFT_INV = 3,  /* inverse FFT, eq. 2.6 (writes the final layout itself when L is a power of two <= 32) */
    NBS_STAGE_OUTPUT = 4,   /* final layout F[ch][a1..a4][r] as a separate pass (other L; else never timed) */
    NBS_NUM_STAGES = 5
};
int nbs_set_timing(nbs_ctx* ctx, int enable);

/*
 * nbs_set_direct -- tiny-lattice path (row a7 of DESIGN.md, the "primitive" O(L^6) evaluation of
 * eq. 2.4): with enable != 0 nbs_correlator takes the zero-momentum sum over X of B1(X+r) B2(X) as a shifted
 * sum in x-space -- the same block, expansion and product kernels, one product task per displacement r that
 * walks all sites X, no FFT.  Results equal the FFT path up to rounding.  Cost O(V^2): NBS_EINVAL for L > 8.
 */
int nbs_set_direct(nbs_ctx* ctx, int enable);

/*
 * nbs_set_pipelined -- which product kernel the resident plan runs (eqs. 4.2-4.3).
 *   enable != 0 (the default whenever it is available): k_product_c -- antisymmetric blocks staged in their compact
 *     form, four block slots in shared memory filled by a host-written load program, warps moving from one sink pair
 *     to the next without a barrier;
 *   enable == 0: k_product_t -- two staged blocks, antisymmetric blocks expanded to full blocks by an extra pass
 *     (a second buffer of nbs_workspace_bytes grows by V * 6 * 6960 * 16 bytes per slot on the first call);
 *   enable < 0: query, returns 1 / 0.
 * Both give the same correlators up to the rounding order of sums of more than two gather terms.  NBS_EINVAL if the
 * pipelined kernel is asked for but the plan has none (fewer than three sink-pair items per momentum pair, tile-wise
 * plan); the tile-wise plan and the direct shifted sum always run k_product_t.  Takes effect at the next nbs_correlator.
 */
int nbs_set_pipelined(nbs_ctx* ctx, int enable);

/*
 * nbs_set_channel_relations -- isospin limit (the caller passed the same array for u and d): besides
 * deriving the blocks of n, Sigma-, Xi- from those of p, Sigma+, Xi0, the library then leaves out every channel of the
 * list that is the u <-> d image of an earlier one and writes it from that one in the epilogue of the product kernel:
 *   <B1 B2 | B3 B4> = eta1 eta2 eta3 eta4 <B1' B2' | B3' B4'>,  <.. | B4' B3'>_{a3 a4} = - <.. | B3' B4'>_{a4 a3},
 * with p <-> n, Sigma+ <-> Sigma-, Xi0 <-> Xi-, X_u <-> X_d (eta = -1 for Lambda, Xi0, Xi-, X_u, X_d, X_s; eqs. 2.2-2.3).
 * In the standard list these are nine channels (n Xi0 -> anything: all six; Lambda Lambda -> n Xi0, Sigma0 Sigma0 ->
 * n Xi0, Sigma0 Lambda -> n Xi0), so the sink pair n Xi0 is not contracted at all.  A sink pair made of a field and its
 * image (p n, Sigma+ Sigma-, Xi- Xi0) is, in addition, contracted for half of the momenta only, like a pair of identical
 * baryons: with the sink swap F^{B1 B2}_{a1 a2}(r) = - F^{B2 B1}_{a2 a1}(-r) the relation above gives
 *   F[B B' | B3 B4](q)_{a1 a2 a3 a4} = - eta eta' eta3 eta4 F[B B' | B3' B4'](-q)_{a2 a1 a3 a4}
 * whenever the channels of the pair are closed under B3 B4 -> B3' B4'.  Results equal the full computation
 * up to rounding.  Resident plan with the pipelined product kernel only.
 *   enable != 0 (default): use the relations;  enable == 0: compute every channel;
 *   enable == -1: query -- returns the number of channels that are derived this way (0: none / not available / off);
 *   enable == -2: query -- the number of sink pairs that are contracted for half of the momenta by the second relation.
 */
int nbs_set_channel_relations(nbs_ctx* ctx, int enable);
/*   nbs_iso_relations: the relations themselves, on the host only (no CUDA call): for channel i of the list (ch == NULL:
 *             the standard 52) from[i] = -1 if it is computed, else F[i] = sign[i] * F[from[i]] with a3 <-> a4 exchanged
 *             if swap34[i]; from[i] < i and channel from[i] is computed.  Writes at most `cap` entries (any array may be
 *             NULL), returns the number of channels, NBS_EINVAL for an invalid baryon id. */
int nbs_iso_relations(const nbs_channel* ch, int nch, int* from, int* sign, int* swap34, int cap);
int nbs_stage_times(nbs_ctx* ctx, double* ms, long long* calls, int reset);

int nbs_exec_flops(const nbs_ctx* ctx, double* product_executed);

/*
 * nbs_probe_fp64 -- FP64 throughput of this device for register-resident instruction mixes (DESIGN.md section 7:
 * the measured denominator of the product kernel's roofline fraction).  Synchronous; runs `iters` iterations of
 *   mode 0: 16 DMMA.8x8x4      mode 1: 16 DFMA      mode 2: 16 DADD
 *   mode 3: 12 DMMA + 12 DADD  (one k-step of the 16x16 accumulator class of the product kernel)
 *   mode 4: 16 DMMA + 24 DADD  (one k-step of the 64x4 class)
 *   mode 5: 12 DADD then 12 DMMA, instruction order pinned      mode 6: DADD and DMMA strictly alternating, order pinned
 *   mode 7 / 8: mode 6 with 8 / 4 independent integer instructions between the FP64 instructions of a pair
 *   (modes 5-8 answer scheduling questions: does interleaving, or integer work in between, cost FP64 throughput)
 * per warp on 16 warps per SM, all SMs.  *tflops = executed FP64 flops per second / 1e12 (a DMMA counts
 * 8*8*4*2 = 512, a DFMA 64, a DADD 32 per warp instruction); *ms = duration of the timed launch.  Either may be NULL.
 */
int nbs_probe_fp64(nbs_ctx* ctx, int mode, int iters, double* tflops, double* ms);

/*
 * nbs_probe_kstep -- the unit code of the pipelined product kernel in isolation (eqs. 4.2-4.3):
 * `warps` warps per SM (1..12; one CTA per SM, 4 sub-partitions) each run the kernel's own device function for the
 * 16x16 accumulator class (cls = 0) or the 64x4 class (cls = 2) `reps` times on a synthetic unit of one diagram with
 * `nsteps` k-steps (1..48): two compact blocks in shared memory, packed gather words read from L2 (another table
 * region every repetition) with the bank-conflict-free offsets the real tables have.  Synchronous.
 * *cycles_per_kstep = SM cycles per k-step of one warp, averaged over all warps (unit prologue and the flush of the
 * 256 results included); divide by warps / 4 for the time a sub-partition needs per k-step and compare with the
 * FP64-pipe time of a k-step from nbs_probe_fp64 (238 / 341 cycles).  *cycles_max = the slowest warp.  Either may be NULL.
 */
int nbs_probe_kstep(nbs_ctx* ctx, int cls, int warps, int nsteps, int reps, double* cycles_per_kstep, double* cycles_max);
int nbs_fft3d(nbs_ctx* ctx, void* data_dev, size_t R, int inverse, void* stream);
long long nbs_kernel_launches(const nbs_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* NBS_H_ */
