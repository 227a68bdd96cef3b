// Generic persistent warp-specialised GEMM core for sm_100a:  D[M,N] = sum_seg A_seg[M,K] * B_seg[N,K]^T
//   TMA (SWIZZLE_128B) -> shared-memory ring -> tcgen05.mma (bf16 -> fp32) -> double-buffered TMEM
//   accumulators -> per-tile epilogue functor run by 4 epilogue warps.
// Two tile configurations of the same code (template parameter CG = tcgen05 cta_group):
//   CG = 1   one CTA per tile, 128 x 256 x 16 MMAs, 4 stages of 48 KiB
//   CG = 2   a CTA pair (cluster of 2, one SM each) per 256 x 256 tile: each CTA loads its own 128 rows of A and
//            its own 128 of B's 256 columns, the pair leader issues 256 x 256 x 16 MMAs that read both CTAs'
//            shared memory and write 128 accumulator rows into each CTA's TMEM; 6 stages of 32 KiB.  Per SM this
//            moves 2/3 of the operand bytes of CG = 1 through L2 -> SMEM and halves the B reads of the MMA.
// A and B may each be K-major (K contiguous in global memory) or MN-major (M/N contiguous); the majorness is a
// run-time parameter that only changes the TMA box sequence and the UMMA descriptors.
// Every GEMM of the OPD path (logits, G re-formation, grad_hidden, grad_W) runs on this core with a different
// epilogue (opd_epilogues.cuh), either as gemm_kernel (one GEMM per launch) or inside bwd_kernel.
#pragma once
#include "opd_ptx.cuh"

namespace opd {

constexpr int BM = 128;              // accumulator rows per CTA (TMEM lanes)
constexpr int BN = 256;              // tile cols   (TMEM columns, fp32)
constexpr int BK = 64;               // bf16 elements per k-block = one 128-byte swizzle row
constexpr int UMMA_K = 16;
constexpr int MN_BOX = 64;                            // MN-major operands arrive as 64(mn) x 64(k) boxes
constexpr int MN_BOX_BYTES = MN_BOX * BK * 2;         // 8 KiB
constexpr int GEMM_THREADS = 192;                     // warp0 TMA, warp1 MMA(+TMEM alloc), warps2-5 epilogue
#ifndef OPD_BWD_EPI_WARPS
#define OPD_BWD_EPI_WARPS 4
#endif
// Epilogue warps of bwd_kernel: 4 (one per TMEM lane quarter), or 8 with -DOPD_BWD_EPI_WARPS=8 (two per quarter, each half of
// a G tile's columns).  8 was measured no faster (the TMEM and LSU ports it would overlap are per SM, not per scheduler) and caps the
// kernel at 168 registers per thread (profiles/r02_trace.md): an experiment, not the product configuration.
constexpr int BWD_EPI_WARPS = OPD_BWD_EPI_WARPS;
static_assert(BWD_EPI_WARPS == 4 || BWD_EPI_WARPS == 8, "one or two epilogue warps per TMEM lane quarter");
constexpr int BWD_THREADS = (2 + BWD_EPI_WARPS + 1) * 32;   // + the publisher of finished tiles (last warp)
constexpr int PUB_Q = 4;                              // tiles the epilogue warps may run ahead of the publisher
constexpr int EPI_SMEM_BYTES = 32768;                 // 4 epilogue warps x 2 staging buffers x (32 rows x 128 B)
constexpr int TMEM_COLS = 512;                        // 2 accumulator stages x 256 columns
constexpr int MAX_STAGES = 6;
// TMA ring depth of the CTA-pair configuration (32 KiB per stage), per kernel (profiles/r02_experiments.md section 3):
//   one-GEMM kernels (forward logits, producers): 4 stages keep the tensor pipe 98% busy and read W from HBM about once per
//     token panel (10.6 GB per C4 launch; 6 stages let the pairs sharing a panel drift apart and re-fetch 46 GB);
//   persistent backward: its operands miss L2 more often (G ring, partial sums, two W panels), 6 stages hide that latency
//     better (tensor pipe 87% against 78% busy).
#ifndef OPD_FWD_STAGES
#define OPD_FWD_STAGES 4
#endif
#ifndef OPD_BWD_STAGES
#define OPD_BWD_STAGES 6
#endif
constexpr int SCHED_Q = 8;                 // depth of the tile queue of the dynamically scheduled kernels
constexpr int SCHED_WORDS = 12;            // 32-bit words of one decoded tile descriptor in the queue (48 bytes)

static_assert(256 + 2 * SCHED_Q * 8 + SCHED_Q * SCHED_WORDS * 4 <= 768 && 768 + 2 * PUB_Q * 8 + PUB_Q * 8 <= 1024, "barrier region is 1 KiB");
template <int CG> __host__ __device__ constexpr int fwd_stages() { return CG == 1 ? 4 : OPD_FWD_STAGES; }
template <int CG> __host__ __device__ constexpr int bwd_stages() { return CG == 1 ? 4 : OPD_BWD_STAGES; }

template <int CG, int ST>
struct Cfg {
    static constexpr int TILE_M = BM * CG;                // rows of one tile (of the CTA or of the pair)
    static constexpr int B_ROWS = BN / CG;                // B rows (n) each CTA loads
    static constexpr int A_STAGE_BYTES = BM * BK * 2;     // 16 KiB
    static constexpr int B_STAGE_BYTES = B_ROWS * BK * 2; // 32 / 16 KiB
    static constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;
    static constexpr int STAGES = ST;
    static constexpr int RING_BYTES = STAGES * STAGE_BYTES;
    static constexpr int SMEM_BYTES = RING_BYTES + 1024 /*barriers*/ + EPI_SMEM_BYTES + 1024 /*align slack*/;
};

enum TokDim { TOK_NONE = 0, TOK_M = 1, TOK_K = 2 };
constexpr int MAX_SEG = 6;

struct GemmParams {
    int M, N, K;              // extents of this GEMM (upper bounds; the token extent is clipped on the device)
    int num_n;                // ceil(N / BN)
    int group_m;              // raster: tiles are walked in groups of group_m row-tiles, m fastest inside
    int a_mn, b_mn;           // 1 = MN-major operand (M/N contiguous in memory), 0 = K-major
    int a_off, b_off;         // M / N element offsets of this GEMM inside the tensors the TMA maps describe
    int ka_off, kb_off;       // K element offsets inside A's and B's tensor
    int nseg;                 // K segments (1 for bf16; 6 for the 3-way bf16 split of fp32 operands)
    unsigned char sa[MAX_SEG], sb[MAX_SEG];   // plane (3rd TMA coordinate) of A / B per segment
    int tok_dim;              // which extent counts live tokens (clipped to n_live - tok_off on the device)
    int tok_off;
    const int* n_live;        // device scalar: number of live tokens (compacted rows)
    // per-launch / per-tile epilogue switches (set by the host for gemm_kernel, per tile by bwd_kernel)
    unsigned long long a_hint, b_hint;   // L2 eviction policy of the operand loads (0 = normal)
    int first, last;          // DxEpi: first / last vocabulary super-tile of this token super-tile
    int row_off, col_off;     // DwEpi: position of this GEMM's output inside grad_W
#ifdef OPD_EXPERIMENTS
    int skip_b;               // TileOp::skip_b of a one-GEMM launch
#endif
#ifdef OPD_TRACE
    long long* tr;            // tracing builds: cycle sums of the epilogue that runs this tile (slot 6: TMEM waits, 7: chunk bodies)
#endif
};

__device__ __forceinline__ void tile_coords(int tile, int num_m, int num_n, int group_m, int& m_blk, int& n_blk) {
    const int per_group = group_m * num_n;
    const int g = tile / per_group;
    const int r = tile - g * per_group;
    const int m0 = g * group_m;
    const int gm = min(group_m, num_m - m0);
    m_blk = m0 + r % gm;
    n_blk = r / gm;
}

// ------------------------------------------------------------------------------------------------ pipeline
// Shared-memory carve-up, barriers and TMEM of one CTA.
//   full[s]    (leader's copy is the live one for CG = 2) TMA bytes of stage s have landed (both CTAs' bytes)
//   empty[s]   the MMAs that read stage s have completed (commit, multicast to both CTAs for CG = 2)
//   tfull[a]   accumulator stage a is complete (commit, multicast)
//   tempty[a]  (leader's copy) all 4*CG epilogue warps have drained accumulator stage a
template <int CG, int ST>
struct Pipe {
    using C = Cfg<CG, ST>;
    uint8_t* smem;
    uint64_t *full_bar, *empty_bar, *tfull_bar, *tempty_bar;
    uint64_t *sfull_bar, *sempty_bar;     // tile queue (bwd_kernel): slot q published / consumed by every reader
    uint32_t* sticket;                    // [SCHED_Q][SCHED_WORDS] decoded tiles (a copy in each CTA of a pair)
    uint64_t *pub_full, *pub_empty;       // publisher queue (bwd_kernel): the 4 epilogue warps are done with tile n / slot reusable
    int** pub_ptr;                        // [PUB_Q] dependency counter the publisher increments for that tile (null: stop)
    uint32_t* tmem_slot;
    uint8_t* epi_smem;
    uint32_t tmem_base;
    uint32_t rank;            // CTA rank in the pair (0 = leader; always 0 for CG = 1)

    __device__ __forceinline__ void setup(uint8_t* smem_raw, int warp, int lane, int epi_warps = 4) {
        smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
        full_bar = reinterpret_cast<uint64_t*>(smem + C::RING_BYTES);
        empty_bar = full_bar + MAX_STAGES;
        tfull_bar = empty_bar + MAX_STAGES;
        tempty_bar = tfull_bar + 2;
        tmem_slot = reinterpret_cast<uint32_t*>(tempty_bar + 2);
        sfull_bar = reinterpret_cast<uint64_t*>(smem + C::RING_BYTES + 256);
        sempty_bar = sfull_bar + SCHED_Q;
        sticket = reinterpret_cast<uint32_t*>(sempty_bar + SCHED_Q);
        pub_full = reinterpret_cast<uint64_t*>(smem + C::RING_BYTES + 768);
        pub_empty = pub_full + PUB_Q;
        pub_ptr = reinterpret_cast<int**>(pub_empty + PUB_Q);
        epi_smem = smem + C::RING_BYTES + 1024;
        rank = CG == 1 ? 0u : cluster_ctarank();
        if (warp == 0 && lane == 0) {
            for (int s = 0; s < C::STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
            for (int s = 0; s < 2; ++s) { mbar_init(&tfull_bar[s], 1); mbar_init(&tempty_bar[s], epi_warps * CG); }
            // readers of a ticket.  CG = 1: the MMA issuer and the epilogue warps (the producer claims).  CG = 2: both
            // producers, the MMA issuer and the epilogue warps of both CTAs of the pair (the peer CTA's otherwise idle warp 1 claims,
            // so that the round trip of the claim never sits between two tiles of the producer)
            for (int s = 0; s < SCHED_Q; ++s) { mbar_init(&sfull_bar[s], 1); mbar_init(&sempty_bar[s], CG == 1 ? 1 + epi_warps : 3 + 2 * epi_warps); }
            for (int s = 0; s < PUB_Q; ++s) { mbar_init(&pub_full[s], epi_warps); mbar_init(&pub_empty[s], 1); }
            fence_mbar_init();
        }
        if (warp == 1) {
            tmem_alloc<CG>(tmem_slot, TMEM_COLS);
            tmem_relinquish<CG>();
        }
        tc_fence_before();
        if constexpr (CG == 1) __syncthreads(); else cluster_sync_all();
        tc_fence_after();
        tmem_base = *tmem_slot;
    }
    __device__ __forceinline__ void teardown(int warp) {
        tc_fence_before();
        if constexpr (CG == 1) __syncthreads(); else cluster_sync_all();   // the peer may still signal our barriers
        if (warp == 1) tmem_dealloc<CG>(tmem_base, TMEM_COLS);
    }
};

// ------------------------------------------------------------------------------------------------ tile queue
// Dynamic tile scheduling for kernels whose tiles wait on tiles of other CTAs: ONE thread of a CTA (pair) claims the next
// item of the tile list from a global counter, DECODES it, and publishes the decoded descriptor (SCHED_WORDS words) to every
// warp role of the CTA (pair) through a small queue in shared memory.  Items are claimed in list order, so everything an
// item depends on has been claimed by a CTA that is already running: the kernel makes progress with any number of resident
// CTAs (no co-residency requirement).  The claimer runs in CTA rank CG - 1 (its copy of the `sempty` barriers is the live
// one), up to SCHED_Q tiles ahead of the slowest reader; readers only copy 48 bytes out of shared memory, so nothing
// but two barrier operations sits between two tiles of the TMA producer or the MMA issuer (the round trip of the global
// atomic and the integer divisions of the decoder are the claimer's: profiles/r02_trace.md).  Only items the launch
// really runs are published (the claimer drops disabled tile types).
__device__ __forceinline__ uint32_t ticket_take(int* counter) { return static_cast<uint32_t>(atomicAdd(counter, 1)); }
__device__ __forceinline__ void st_shared_cluster_v4(uint32_t cluster_addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared::cluster.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(cluster_addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
template <int CG, int ST>
__device__ __forceinline__ void tile_publish(const Pipe<CG, ST>& P, int n, const uint32_t (&w)[SCHED_WORDS]) {
    const int q = n % SCHED_Q;
    mbar_wait_cluster(&P.sempty_bar[q], ((n / SCHED_Q) & 1) ^ 1);
    uint32_t* slot = P.sticket + q * SCHED_WORDS;
#pragma unroll
    for (int i = 0; i < SCHED_WORDS; i += 4) *reinterpret_cast<uint4*>(slot + i) = make_uint4(w[i], w[i + 1], w[i + 2], w[i + 3]);
    if constexpr (CG == 2) {
        const uint32_t remote = mapa_rank(smem_u32(slot), 0);
#pragma unroll
        for (int i = 0; i < SCHED_WORDS; i += 4) st_shared_cluster_v4(remote + i * 4, w[i], w[i + 1], w[i + 2], w[i + 3]);
        mbar_arrive_cluster(mapa_rank(smem_u32(&P.sfull_bar[q]), 0));
    }
    mbar_arrive(&P.sfull_bar[q]);
}
// Called by one thread of a reader (wait = true) and, for warp-wide readers, by the other lanes after a __syncwarp
// (wait = false); every reader consumes every slot exactly once, in order, and signals it with tile_consumed.
template <int CG, int ST>
__device__ __forceinline__ void tile_wait(const Pipe<CG, ST>& P, int n) {
    mbar_wait_cluster(&P.sfull_bar[n % SCHED_Q], (n / SCHED_Q) & 1);
}
template <int CG, int ST>
__device__ __forceinline__ void tile_copy(const Pipe<CG, ST>& P, int n, uint32_t (&w)[SCHED_WORDS]) {
    const volatile uint4* slot = reinterpret_cast<const volatile uint4*>(P.sticket + (n % SCHED_Q) * SCHED_WORDS);
#pragma unroll
    for (int i = 0; i < SCHED_WORDS / 4; ++i) {
        w[4 * i] = slot[i].x; w[4 * i + 1] = slot[i].y; w[4 * i + 2] = slot[i].z; w[4 * i + 3] = slot[i].w;
    }
}
template <int CG, int ST>
__device__ __forceinline__ void tile_consumed(const Pipe<CG, ST>& P, int n) {
    mbar_arrive_remote(mapa_rank(smem_u32(&P.sempty_bar[n % SCHED_Q]), CG - 1));     // a read-done signal: no cluster release
}

// One tile's operand stream as the TMA producer of ONE CTA sees it.
struct TileOp {
    const CUtensorMap* tA;
    const CUtensorMap* tB;
    int a_mn, b_mn;
    int a_c, b_c;             // first M row of A / first N row of B this CTA loads
    int ka, kb;               // K offsets
    int K;
    int nseg;
    unsigned char pa[MAX_SEG], pb[MAX_SEG];   // plane per segment
    uint64_t a_hint, b_hint;  // L2 eviction policy of the operand loads
#ifdef OPD_EXPERIMENTS
    int skip_b = 0;           // timing experiment (wrong results): after the first ring fill the B operand is not loaded any more
#endif
};

// TMA producer (one elected lane): stream all k-blocks of all segments of `t` through the ring.
struct NoMid { __device__ __forceinline__ void operator()() const {} };

// `mid` runs once, after the loads of the tile's second k-block have been issued (after the last one for shorter tiles): the
// persistent kernels fetch and decode their NEXT tile there, while the ring still holds work for the tensor pipe.
// Tracing builds (-DOPD_TRACE, profiles/r02_trace.md): `tr` accumulates the cycles a role spends in its waits.
template <int CG, int ST, class Mid = NoMid>
__device__ __forceinline__ void produce_tile(const Pipe<CG, ST>& P, const TileOp& t, int& it, Mid&& mid = Mid{}, long long* tr = nullptr) {
    using C = Cfg<CG, ST>;
    const int kblocks = (t.K + BK - 1) / BK;
    const int mid_at = min(2, kblocks * t.nseg);
    int issued = 0;
    for (int seg = 0; seg < t.nseg; ++seg) {
        for (int kb_i = 0; kb_i < kblocks; ++kb_i, ++it) {
#ifdef OPD_TRACE
            if (issued++ == mid_at) { const long long t0 = clock64(); mid(); if (tr) tr[4] += clock64() - t0; }
            const int s = it % C::STAGES;
            const uint32_t ph = (it / C::STAGES) & 1;
            if (tr) mbar_wait_timed(&P.empty_bar[s], ph ^ 1, tr[2]); else mbar_wait(&P.empty_bar[s], ph ^ 1);
#else
            if (issued++ == mid_at) mid();
            const int s = it % C::STAGES;
            const uint32_t ph = (it / C::STAGES) & 1;
            mbar_wait(&P.empty_bar[s], ph ^ 1);
#endif
            uint8_t* sA = P.smem + s * C::STAGE_BYTES;
            uint8_t* sB = sA + C::A_STAGE_BYTES;
            const int kca = t.ka + kb_i * BK, kcb = t.kb + kb_i * BK;
            const int pa = t.pa[seg], pb = t.pb[seg];
            if constexpr (CG == 1) {
                uint64_t* bar = &P.full_bar[s];
                mbar_arrive_expect_tx(bar, C::STAGE_BYTES);
                if (t.a_mn) {
                    for (int b = 0; b < BM / MN_BOX; ++b) tma_load_3d(sA + b * MN_BOX_BYTES, t.tA, bar, t.a_c + b * MN_BOX, kca, pa, t.a_hint);
                } else {
                    tma_load_3d(sA, t.tA, bar, kca, t.a_c, pa, t.a_hint);
                }
                if (t.b_mn) {
                    for (int b = 0; b < C::B_ROWS / MN_BOX; ++b) tma_load_3d(sB + b * MN_BOX_BYTES, t.tB, bar, t.b_c + b * MN_BOX, kcb, pb, t.b_hint);
                } else {
                    tma_load_3d(sB, t.tB, bar, kcb, t.b_c, pb, t.b_hint);
                }
            } else {
                // the leader's barrier counts the bytes of both CTAs (expect_tx may trail the peer's complete_tx:
                // the phase cannot complete before the leader's own arrival)
#ifdef OPD_EXPERIMENTS
                const bool skipb = t.skip_b && it >= C::STAGES;
#else
                constexpr bool skipb = false;
#endif
                if (P.rank == 0) mbar_arrive_expect_tx(&P.full_bar[s], skipb ? 2 * C::A_STAGE_BYTES : 2 * C::STAGE_BYTES);
                const uint32_t bar = mapa_rank(smem_u32(&P.full_bar[s]), 0);
                if (t.a_mn) {
                    for (int b = 0; b < BM / MN_BOX; ++b) tma_load_3d_pair(sA + b * MN_BOX_BYTES, t.tA, bar, t.a_c + b * MN_BOX, kca, pa, t.a_hint);
                } else {
                    tma_load_3d_pair(sA, t.tA, bar, kca, t.a_c, pa, t.a_hint);
                }
                if (skipb) {
                } else if (t.b_mn) {
                    for (int b = 0; b < C::B_ROWS / MN_BOX; ++b) tma_load_3d_pair(sB + b * MN_BOX_BYTES, t.tB, bar, t.b_c + b * MN_BOX, kcb, pb, t.b_hint);
                } else {
                    tma_load_3d_pair(sB, t.tB, bar, kcb, t.b_c, pb, t.b_hint);
                }
            }
        }
    }
    if (issued <= mid_at) mid();
}

// MMA issuer (one elected lane of the CTA / of the pair leader): all MMAs of one tile into accumulator stage lt & 1.
template <int CG, int ST, class Mid = NoMid>
__device__ __forceinline__ void mma_tile(const Pipe<CG, ST>& P, int a_mn, int b_mn, int kiters, int lt, int& it, Mid&& mid = Mid{}, long long* tr = nullptr) {
    using C = Cfg<CG, ST>;
    const uint32_t idesc = make_idesc_bf16(C::TILE_M, BN, a_mn, b_mn);
    const uint32_t a_kstep = a_mn ? (UMMA_K * MN_BOX * 2) : (UMMA_K * 2);   // bytes per UMMA_K step
    const uint32_t b_kstep = b_mn ? (UMMA_K * MN_BOX * 2) : (UMMA_K * 2);
    const uint32_t a_lbo = a_mn ? MN_BOX_BYTES : 16;
    const uint32_t b_lbo = b_mn ? MN_BOX_BYTES : 16;
    const int as = lt & 1;
    const uint32_t aph = (lt >> 1) & 1;
#ifdef OPD_TRACE
    if (tr) mbar_wait_timed(&P.tempty_bar[as], aph ^ 1, tr[2]); else
#endif
    mbar_wait(&P.tempty_bar[as], aph ^ 1);
    tc_fence_after();
    const uint32_t tacc = P.tmem_base + as * BN;
    // `mid` (the persistent kernels read their next tile there) runs where the issuer would block anyway: the ring's
    // stages have all been issued and the next one only fills once the tensor pipe has retired this tile's first k-block
    const int mid_at = min(C::STAGES, kiters - 1);
    for (int ki = 0; ki < kiters; ++ki, ++it) {
#ifdef OPD_TRACE
        if (ki == mid_at) { const long long t0 = clock64(); mid(); if (tr) tr[4] += clock64() - t0; }
        const int s = it % C::STAGES;
        const uint32_t ph = (it / C::STAGES) & 1;
        if (tr) mbar_wait_timed(&P.full_bar[s], ph, tr[ki < C::STAGES ? 5 : 3]); else mbar_wait(&P.full_bar[s], ph);
#else
        if (ki == mid_at) mid();                   // MMAs of the first k-blocks are queued: time to decode the next tile
        const int s = it % C::STAGES;
        const uint32_t ph = (it / C::STAGES) & 1;
        mbar_wait(&P.full_bar[s], ph);
#endif
        tc_fence_after();
        const uint32_t a0 = smem_u32(P.smem + s * C::STAGE_BYTES);
        const uint32_t b0 = a0 + C::A_STAGE_BYTES;
#pragma unroll
        for (int k = 0; k < BK / UMMA_K; ++k) {
            const uint64_t ad = make_smem_desc(a0 + k * a_kstep, a_lbo, 1024);
            const uint64_t bd = make_smem_desc(b0 + k * b_kstep, b_lbo, 1024);
            umma_bf16<CG>(tacc, ad, bd, idesc, (ki | k) != 0);
        }
        umma_commit<CG>(&P.empty_bar[s]);          // frees the smem slot (in both CTAs) once these MMAs have read it
    }
    umma_commit<CG>(&P.tfull_bar[as]);             // accumulator complete -> epilogue warps (of both CTAs)
}

// Epilogue side: wait for accumulator stage lt & 1; returns this warp's TMEM address (lane quarter in bits 16+).
template <int CG, int ST>
__device__ __forceinline__ uint32_t epi_acquire(const Pipe<CG, ST>& P, int lt, int quarter) {
    const int as = lt & 1;
    mbar_wait(&P.tfull_bar[as], (lt >> 1) & 1);
    tc_fence_after();
    return P.tmem_base + as * BN + (static_cast<uint32_t>(quarter * 32) << 16);
}
template <int CG, int ST>
__device__ __forceinline__ void epi_release(const Pipe<CG, ST>& P, int lt, int lane) {
    tc_fence_before();
    __syncwarp();
    if (lane == 0) {
        if constexpr (CG == 1) mbar_arrive(&P.tempty_bar[lt & 1]);
        else mbar_arrive_remote(mapa_rank(smem_u32(&P.tempty_bar[lt & 1]), 0));      // read-done signal (see mbar_arrive_remote)
    }
}

// ------------------------------------------------------------------------------------------------ one GEMM per launch
// Epi must provide:  struct Params;  struct State;  static State prepare(...);
//                    static void run(const Params&, const GemmParams&, State, uint32_t taddr, int m_blk, int n_blk,
//                                    int row_in_tile, int M_eff, uint8_t* epi_smem, int epi_tid)
// with m_blk counting 128-row blocks (for CG = 2 the pair's tile is row blocks 2*m2 and 2*m2 + 1).
template <class Epi, int CG>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
            const GemmParams gp, const __grid_constant__ typename Epi::Params ep) {
    constexpr int ST = fwd_stages<CG>();
    using C = Cfg<CG, ST>;
    extern __shared__ uint8_t smem_raw[];
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    // ---- device-side extents (the live-token count is only known on the device)
    int M = gp.M, K = gp.K;
    if (gp.tok_dim != TOK_NONE) {
        const int live = *gp.n_live - gp.tok_off;
        if (gp.tok_dim == TOK_M) M = min(M, live);
        else K = min(K, live);
    }
    if (M <= 0 || K <= 0) return;                     // uniform over the grid
    const int num_m = (M + C::TILE_M - 1) / C::TILE_M;
    const int num_n = gp.num_n;
    const int total_tiles = num_m * num_n;
    const int kblocks = (K + BK - 1) / BK;
    const int first_tile = blockIdx.x / CG, tile_step = gridDim.x / CG;

    if (warp == 0 && lane == 0) { prefetch_tmap(&tmA); prefetch_tmap(&tmB); }
    Pipe<CG, ST> P;
    P.setup(smem_raw, warp, lane);

    if (warp == 0) {
        // =========================== TMA producer (one elected lane) ===========================
        if (elect_one()) {
            TileOp t;
            t.tA = &tmA; t.tB = &tmB; t.a_mn = gp.a_mn; t.b_mn = gp.b_mn; t.ka = gp.ka_off; t.kb = gp.kb_off; t.K = K;
            t.nseg = gp.nseg;
            t.a_hint = gp.a_hint ? gp.a_hint : L2_EVICT_NORMAL; t.b_hint = gp.b_hint ? gp.b_hint : L2_EVICT_NORMAL;
            for (int i = 0; i < MAX_SEG; ++i) { t.pa[i] = gp.sa[i]; t.pb[i] = gp.sb[i]; }
#ifdef OPD_EXPERIMENTS
            t.skip_b = gp.skip_b;
#endif
            int it = 0;
            for (int tile = first_tile; tile < total_tiles; tile += tile_step) {
                int m2, n_blk;
                tile_coords(tile, num_m, num_n, gp.group_m, m2, n_blk);
                t.a_c = gp.a_off + (m2 * CG + static_cast<int>(P.rank)) * BM;
                t.b_c = gp.b_off + n_blk * BN + static_cast<int>(P.rank) * C::B_ROWS;
                produce_tile<CG, ST>(P, t, it);
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer (one elected lane of the leader) ===========================
        if (P.rank == 0 && elect_one()) {
            int it = 0, lt = 0;
            for (int tile = first_tile; tile < total_tiles; tile += tile_step, ++lt)
                mma_tile<CG, ST>(P, gp.a_mn, gp.b_mn, kblocks * gp.nseg, lt, it);
        }
    } else {
        // =========================== epilogue warps (TMEM -> registers -> global) ===========================
        const int quarter = warp & 3;                    // TMEM lane quarter this warp may access
        const int row_in_tile = quarter * 32 + lane;
        const int epi_tid = (warp - 2) * 32 + lane;
        int lt = 0;
        for (int tile = first_tile; tile < total_tiles; tile += tile_step, ++lt) {
            int m2, n_blk;
            tile_coords(tile, num_m, num_n, gp.group_m, m2, n_blk);
            const int m_blk = m2 * CG + static_cast<int>(P.rank);
            // per-row state (scalars, cache cursor) is fetched while the MMAs of this tile are still running
            typename Epi::State st = Epi::prepare(ep, gp, m_blk, n_blk, row_in_tile, M);
            const uint32_t taddr = epi_acquire<CG, ST>(P, lt, quarter);
            Epi::run(ep, gp, st, taddr, m_blk, n_blk, row_in_tile, M, P.epi_smem, epi_tid);
            epi_release<CG, ST>(P, lt, lane);
        }
    }
    P.teardown(warp);
}

}  // namespace opd
