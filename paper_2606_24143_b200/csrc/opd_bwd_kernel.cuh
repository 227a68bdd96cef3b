// One persistent kernel for the whole backward (S6-S8).  Same warp-specialised tcgen05 pipeline as
// gemm_kernel, but the tile list interleaves three GEMM kinds over all (token x vocabulary) super-tiles:
//
//   block 0: G(0)      block b: G(b), DX(b-1), DW(b-1)      block S: DX(S-1), DW(S-1)
//
//   G(s)   logits of super-tile s recomputed -> G tile (bf16) into buffer s%R of the G ring (consumed from L2)
//   DX(s)  grad_hidden[tb] (+)= G(s) . W[:,vb]^T        DW(s)  grad_W[:,vb] += Xc[tb]^T . G(s)
//
// CTA pairs claim items dynamically, in list order, from a global ticket counter (the tile queue of opd_gemm.cuh: one thread
// per pair claims, decodes and publishes the tile, every warp role copies it); an item only depends on earlier items,
// through three counters per super-tile in global memory (release by the publisher warp once the epilogue's stores are out,
// acquire by whoever consumes):
//   g_done[s] == #G tiles          before the TMA producer loads G(s) for a DX/DW tile
//   dx_done[s-1] complete          before a DX(s) epilogue touches the fp32 partial sums of grad_hidden (previous writer; at a
//                                  token super-tile boundary: the previous reader)
//   dw_done[s-nvb] complete        before a DW(s) epilogue reduces into its grad_W panel (previous token super-tile, same columns)
//   dx_done, dw_done[s-R] complete before a G(s) epilogue overwrites ring buffer s%R (previous readers; R = ring depth)
// (one counter for DX and DW made every DX(s) epilogue wait for the long DW(s-1) tiles that were claimed just before it and
// share nothing with it: 18% of the epilogue warps' time at T = 4096, d = 1024.)
// One launch instead of one per GEMM and super-tile (about 900 at C4): no partial last waves, no pipeline refills.
// Because an item's dependencies were all claimed before it, by CTAs that are running, the kernel needs no particular
// number of resident CTAs: it completes next to other kernels, under MPS or with SM-limited contexts (the host still sizes
// the grid to one CTA per SM, which is the fastest configuration).  The order in which tiles are reduced into an fp32
// accumulator is fixed by the counters, not by which CTA runs a tile: results stay bit-reproducible.
#pragma once
#include "opd_dense.cuh"

namespace opd {

struct BwdParams {
    int d, V, Tb, Vb, nvb;     // super-tile rows / cols, vocabulary super-tiles per token super-tile
    int wl;                    // 0: W is [d,V] row-major, 1: [V,d]
    int gbufs;                 // depth of the G ring (2 or 3)
    int planes;                // 1 (bf16) or 3 (fp32 inputs as three bf16 terms)
    const int* n_live;
    int* g_done;               // [S]
    int* dx_done;              // [S]
    int* dw_done;              // [S]
    int* ticket;               // [1] next unclaimed item of the tile list (zeroed by the host before the launch)
    int order;                 // BwdSched::order
    int q_depth;               // tiles a CTA (pair) may hold claimed but not yet started by its epilogue (1..SCHED_Q)
    int dx_group;              // BwdSched::dx_group
    int dw_store_first;        // 1: the grad_W tiles of the first token super-tile store instead of reduce-add (grad_W is
                               //    overwritten, not accumulated into: no memset and no read-modify-write for that pass)
    int type_mask;             // bit t set = run tiles of type t.  All types of the variant = the normal run; a tile waits
                               // on a counter only if every tile type that increments it is enabled (dense forward-only
                               // runs Q + G; other subsets are timing experiments and give wrong gradients)
    unsigned long long hint_x, hint_w, hint_g;   // L2 eviction policies of the Xc / W / G-ring operand loads
    GEpi::Params g;            // gs points at ring buffer 0; buffer b at + b * planes * plane_stride
    DxEpi::Params dx;
    DwEpi::Params dw;
    // dense two-head variant (opd_dense.cuh): teacher contraction depth / layout, Q ring and its counter
    int dT, wl_t, qbytes;      // qbytes: element size of the Q ring (2 bf16, 4 fp32)
    int* q_done;               // [S]
    QEpi::Params q;            // qs points at Q ring buffer 0; buffer b at + b * q_buf_bytes
    size_t q_buf_bytes;
    GDenseEpi::Params gd;
#ifdef OPD_TRACE
    unsigned long long* trace; // [3 roles][4 tile types][8] cycle sums + [96..] per-CTA kernel cycles (tracing builds only)
#endif
};

enum { T_G = 0, T_DX = 1, T_DW = 2, T_Q = 3 };

// One decoded item of the tile list: what the claimer publishes through the tile queue (SCHED_WORDS words).
struct BwdTile {
    int type, s, tb0, vb0, Tb_eff, Vb_eff, vi, m_blk, n_blk;
    int ng;                    // G tiles of super-tile s (what a DX / DW tile waits for)
    int dep_cnt;               // CTA-level epilogues the counter(s) this tile's epilogue waits on must have seen (0: no wait):
                               //   DX: dx_done[s - 1]; DW: dw_done[s - nvb]; G: dx_done[s - R] in the low and dw_done[s - R] in the
                               //   high 16 bits; Q (dense): g_done[s - 2]
    int valid;                 // 0: the list is exhausted (published once, every reader stops on it)
};
static_assert(sizeof(BwdTile) == SCHED_WORDS * 4, "BwdTile is what the tile queue carries");

// DENSE: block b holds Q(b), G(b-1), DX(b-2), DW(b-2) (the Q tiles of a super-tile run one block ahead of its G tiles);
// otherwise block b holds G(b), DX(b-1), DW(b-1).
// The decoder keeps the tile counts and extents of the current block's super-tiles (one integer division per new block),
// so that decoding an item costs a few compares and one division: every warp role decodes every item of its CTA, the MMA
// issuer between two tiles (while the tensor pipe drains its queue).
template <int CG, bool DENSE>
struct BwdSched {
    static constexpr int GOFF = DENSE ? 1 : 0;
    static constexpr int TM = BM * CG;
    struct Super { int s, ti, vi, tb_eff, vb_eff, mt, nt, ng, ndx, ndw; };
    int S, nvb, Tb, Vb, V, d, wl, n_live, dm, dn;
    int order;      // tile order knobs (result-neutral): bit 0 grad_W tiles before grad_hidden tiles inside a block,
                    // bits 1-3: n-fastest raster of the G / grad_hidden / grad_W tiles (default m fastest),
                    // bit 4: G tiles of a block split around its DX / DW tiles (default: all G tiles first)
    int dx_group;   // row tiles per raster group of the grad_hidden tiles (0: all rows of the super-tile)
    int blk;        // current block
    long base;      // items before the current block
    int sz;         // items of the current block
    Super q, g, c;  // super-tiles whose Q / G / (DX, DW) tiles the current block holds (s = -1: none)
    __device__ __forceinline__ void super_info(int s, Super& o) const {
        o.s = s;
        if (s < 0 || s >= S) { o.s = -1; o.ng = o.ndx = o.ndw = 0; return; }
        o.ti = s / nvb; o.vi = s - o.ti * nvb;
        o.tb_eff = min(Tb, n_live - o.ti * Tb);
        o.vb_eff = min(Vb, V - o.vi * Vb);
        o.mt = (o.tb_eff + TM - 1) / TM;
        o.nt = (o.vb_eff + BN - 1) / BN;
        o.ng = o.mt * o.nt;
        o.ndx = o.mt * dn;
        o.ndw = wl == 0 ? dm * o.nt : ((o.vb_eff + TM - 1) / TM) * dn;
    }
    __device__ __forceinline__ void load_block() {
        if (DENSE) super_info(blk, q); else { q.s = -1; q.ng = 0; }
        super_info(blk - GOFF, g);
        super_info(blk - GOFF - 1, c);
        sz = q.ng + g.ng + c.ndx + c.ndw;
    }
    __device__ __forceinline__ void init(const BwdParams& p) {
        n_live = *p.n_live;
        nvb = p.nvb; Tb = p.Tb; Vb = p.Vb; V = p.V; d = p.d; wl = p.wl; order = p.order; dx_group = p.dx_group;
        dm = (d + TM - 1) / TM; dn = (d + BN - 1) / BN;
        S = ((n_live + Tb - 1) / Tb) * nvb;
        blk = 0; base = 0;
        load_block();
    }
    // tile counts (a tile = one CTA's or one CTA pair's TM x 256 output block)
    __device__ __forceinline__ int nG(int s) const { Super o; super_info(s, o); return o.ng; }
    __device__ __forceinline__ int nDX(int s) const { Super o; super_info(s, o); return o.ndx; }
    __device__ __forceinline__ int nDW(int s) const { Super o; super_info(s, o); return o.ndw; }
    // decode `item` (monotonically increasing between calls); false when the list is exhausted
    __device__ __forceinline__ bool get(long item, BwdTile& t) {
        if (S <= 0) return false;
        while (blk <= S + GOFF && item >= base + sz) {
            base += sz; ++blk;
            if (blk <= S + GOFF) {                   // shift: the next block's (DX, DW) super-tile is this block's G super-tile
                if (DENSE) { c = g; g = q; super_info(blk, q); } else { c = g; super_info(blk, g); }
                sz = q.ng + g.ng + c.ndx + c.ndw;
            }
        }
        if (blk > S + GOFF) return false;
        int r = static_cast<int>(item - base);
        const Super* u;
        // order bit 4 (experiment, measured neutral at C4 and 6-7% slower at C2 / C3, profiles/r02_experiments.md): the G tiles
        // of a block split around its DX / DW tiles, [G first half, DX, DW, G second half], so that half a super-tile of G
        // tiles lies between any tile and the tiles it waits for at the block boundaries
        const int gh = (!DENSE && (order & 16)) ? (g.ng + 1) / 2 : g.ng;
        if (DENSE && r < q.ng) { t.type = T_Q; u = &q; }
        else if ((r -= q.ng) < gh) { t.type = T_G; u = &g; }
        else if (r - gh < c.ndx + c.ndw) {
            r -= gh; u = &c;
            if (order & 1) { if (r < c.ndw) t.type = T_DW; else { t.type = T_DX; r -= c.ndw; } }
            else { if (r < c.ndx) t.type = T_DX; else { t.type = T_DW; r -= c.ndx; } }
        } else { r -= c.ndx + c.ndw; t.type = T_G; u = &g; }
        t.s = u->s; t.vi = u->vi; t.Tb_eff = u->tb_eff; t.Vb_eff = u->vb_eff; t.ng = u->ng;
        t.tb0 = u->ti * Tb; t.vb0 = u->vi * Vb;
        const int rows = t.type == T_DW ? (wl == 0 ? dm : (u->vb_eff + TM - 1) / TM) : u->mt;
        const int tbit = t.type == T_DX ? 4 : (t.type == T_DW ? 8 : 2);
        if (order & tbit) {                          // n fastest: concurrently running CTAs share the A panel
            const int cols = t.type == T_DX ? dn : (t.type == T_DW ? (wl == 0 ? u->nt : dn) : u->nt);
            t.m_blk = r / cols; t.n_blk = r - t.m_blk * cols;
        } else if (t.type == T_DX && dx_group > 0 && dx_group < rows) {
            // grad_hidden tiles in groups of dx_group row tiles, m fastest inside a group: the G row panels of one group
            // (dx_group x Vb x 512 bytes) stay in L2 while the W slices stream past, instead of all of G per wave
            const int per_group = dx_group * dn;
            const int gi = r / per_group;
            const int rr = r - gi * per_group;
            const int gm = min(dx_group, rows - gi * dx_group);
            t.n_blk = rr / gm; t.m_blk = gi * dx_group + (rr - t.n_blk * gm);
        } else {                                     // m fastest: concurrently running CTAs share the B panel
            t.n_blk = r / rows; t.m_blk = r - t.n_blk * rows;
        }
        return true;
    }
};

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void wait_counter(const int* c, int expected) {
    while (ld_acquire_gpu(c) < expected) __nanosleep(128);
}
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

// Counters count CTA-level epilogues: a tile of a CTA pair (CG = 2) contributes 2.
// DENSE adds the teacher-head Q tiles of the dense two-head KL (opd_dense.cuh); m_tx_k / m_wt_fwd are then the teacher's
// compacted hidden states and head (unused copies of the student's maps otherwise).
template <int CG, bool DENSE>
__global__ void __launch_bounds__(BWD_THREADS, 1)
bwd_kernel(const __grid_constant__ CUtensorMap m_xc_k, const __grid_constant__ CUtensorMap m_w_fwd,
           const __grid_constant__ CUtensorMap m_gs_k, const __grid_constant__ CUtensorMap m_w_dx,
           const __grid_constant__ CUtensorMap m_xc_mn, const __grid_constant__ CUtensorMap m_gs_mn,
           const __grid_constant__ CUtensorMap m_tx_k, const __grid_constant__ CUtensorMap m_wt_fwd,
           const __grid_constant__ BwdParams bp) {
    constexpr int ST = bwd_stages<CG>();
    using C = Cfg<CG, ST>;
    extern __shared__ uint8_t smem_raw[];
    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    if (*bp.n_live <= 0) return;                      // uniform over the grid

    if (warp == 0 && lane == 0) {
        prefetch_tmap(&m_xc_k); prefetch_tmap(&m_w_fwd); prefetch_tmap(&m_gs_k);
        prefetch_tmap(&m_w_dx); prefetch_tmap(&m_xc_mn); prefetch_tmap(&m_gs_mn);
        if constexpr (DENSE) { prefetch_tmap(&m_tx_k); prefetch_tmap(&m_wt_fwd); }
    }
    Pipe<CG, ST> P;
    P.setup(smem_raw, warp, lane, BWD_EPI_WARPS);
    const int rank = static_cast<int>(P.rank);
    const int mask = bp.type_mask;
    auto on = [mask](int type) { return ((mask >> type) & 1) != 0; };

    // segment tables of the three-term split (planes == 3), see set_segments()
    const int nseg = bp.planes == 1 ? 1 : 6;
    const int PA[6] = {1, 2, 0, 1, 0, 0};      // smallest products first (set_segments)
    const int PB[6] = {1, 0, 2, 0, 1, 0};

    // ---- tile queue.  The claimer takes the next item of the list, decodes it (BwdSched: the integer divisions live here)
    // and publishes the decoded tile; every other role copies 48 bytes out of shared memory.
    auto claim_next = [&](BwdSched<CG, DENSE>& sc, int& n, BwdTile& o) -> bool {
        // A ticket is only taken once the tile q_depth places back has been picked up by every reader of this pair: tiles
        // claimed far ahead sit in this pair's queue while other pairs wait for them (G tiles behind a long grad_W tile).
        if (n >= bp.q_depth) { const int m = n - bp.q_depth; mbar_wait_cluster(&P.sempty_bar[m % SCHED_Q], (m / SCHED_Q) & 1); }
        for (;;) {
            const uint32_t item = ticket_take(bp.ticket);
            const bool ok = sc.get(item, o);
            if (ok && !on(o.type)) continue;             // tile types this launch does not run are never published
            o.valid = ok ? 1 : 0;
            o.dep_cnt = 0;
            if (ok) {
                if (DENSE && o.type == T_Q) {
                    if (o.s >= 2 && on(T_G)) o.dep_cnt = CG * sc.nG(o.s - 2);
                } else if (o.type == T_G) {
                    const int dep = o.s - bp.gbufs;
                    if (dep >= 0 && on(T_DX) && on(T_DW)) o.dep_cnt = (CG * sc.nDX(dep)) | ((CG * sc.nDW(dep)) << 16);
                } else if (o.type == T_DX) {
                    if (o.s >= 1 && on(T_DX)) o.dep_cnt = CG * sc.nDX(o.s - 1);
                } else {
                    if (o.s >= bp.nvb && on(T_DW)) o.dep_cnt = CG * sc.nDW(o.s - bp.nvb);
                }
            }
            tile_publish<CG, ST>(P, n++, reinterpret_cast<const uint32_t(&)[SCHED_WORDS]>(o));
            return ok;                                   // the end of the list is published too: every reader stops on it
        }
    };
#ifdef OPD_TRACE
    long long q_wait = 0, q_copy = 0, q_arrive = 0;      // this thread's cycles in the three steps of read_next
#endif
    auto read_next = [&](int& n, BwdTile& o) -> bool {   // single-thread readers (TMA producer, MMA issuer)
#ifdef OPD_TRACE
        const long long c0 = clock64();
        tile_wait<CG, ST>(P, n);
        const long long c1 = clock64();
        tile_copy<CG, ST>(P, n, reinterpret_cast<uint32_t(&)[SCHED_WORDS]>(o));
        const long long c2 = clock64();
        tile_consumed<CG, ST>(P, n);
        const long long c3 = clock64();
        q_wait += c1 - c0; q_copy += c2 - c1; q_arrive += c3 - c2;
#else
        tile_wait<CG, ST>(P, n);
        tile_copy<CG, ST>(P, n, reinterpret_cast<uint32_t(&)[SCHED_WORDS]>(o));
        tile_consumed<CG, ST>(P, n);
#endif
        ++n;
        return o.valid != 0;
    };

    if (warp == 0) {
        // =========================== TMA producer ===========================
        if (elect_one()) {
            BwdSched<CG, DENSE> sc;
            if constexpr (CG == 1) sc.init(bp);              // CG = 1: the producer is the claimer
            BwdTile t, nxt;
            int it = 0, n = 0, g_ready = -1;
            auto fetch = [&](BwdTile& o) -> bool {
                if constexpr (CG == 1) return claim_next(sc, n, o); else return read_next(n, o);
            };
#ifdef OPD_TRACE
            long long trp[4][8] = {};
            const long long k0 = clock64();
#endif
            bool have = fetch(t), have_next = false;
            while (have) {
#ifdef OPD_TRACE
                long long* tr = trp[t.type];
                const long long t0 = clock64();
#endif
                TileOp op;
                int pa_off = 0, pb_off = 0;
                const int buf = t.s % bp.gbufs;
                const int a_row = (t.m_blk * CG + rank) * BM, b_row = t.n_blk * BN + rank * C::B_ROWS;
                if (t.type == T_G) {
                    op.tA = &m_xc_k; op.tB = &m_w_fwd; op.a_mn = 0; op.b_mn = (bp.wl == 0);
                    op.a_c = t.tb0 + a_row; op.b_c = t.vb0 + b_row; op.ka = 0; op.kb = 0; op.K = bp.d;
                    op.a_hint = bp.hint_x; op.b_hint = bp.hint_w;
                } else if (DENSE && t.type == T_Q) {
                    op.tA = &m_tx_k; op.tB = &m_wt_fwd; op.a_mn = 0; op.b_mn = (bp.wl_t == 0);
                    op.a_c = t.tb0 + a_row; op.b_c = t.vb0 + b_row; op.ka = 0; op.kb = 0; op.K = bp.dT;
                    op.a_hint = bp.hint_x; op.b_hint = bp.hint_w;
                } else if (t.type == T_DX) {
                    op.tA = &m_gs_k; op.tB = &m_w_dx; op.a_mn = 0; op.b_mn = (bp.wl == 1);
                    op.a_c = a_row; op.b_c = b_row; op.ka = 0; op.kb = t.vb0; op.K = t.Vb_eff; pa_off = buf * bp.planes;
                    op.a_hint = bp.hint_g; op.b_hint = bp.hint_w;
                } else if (bp.wl == 0) {
                    op.tA = &m_xc_mn; op.tB = &m_gs_mn; op.a_mn = 1; op.b_mn = 1;
                    op.a_c = a_row; op.b_c = b_row; op.ka = t.tb0; op.kb = 0; op.K = t.Tb_eff; pb_off = buf * bp.planes;
                    op.a_hint = bp.hint_x; op.b_hint = bp.hint_g;
                } else {
                    op.tA = &m_gs_mn; op.tB = &m_xc_mn; op.a_mn = 1; op.b_mn = 1;
                    op.a_c = a_row; op.b_c = b_row; op.ka = 0; op.kb = t.tb0; op.K = t.Tb_eff; pa_off = buf * bp.planes;
                    op.a_hint = bp.hint_g; op.b_hint = bp.hint_x;
                }
                op.nseg = nseg;
                for (int i = 0; i < nseg; ++i) {
                    op.pa[i] = static_cast<unsigned char>(pa_off + (nseg == 1 ? 0 : PA[i]));
                    op.pb[i] = static_cast<unsigned char>(pb_off + (nseg == 1 ? 0 : PB[i]));
                }
                if ((t.type == T_DX || t.type == T_DW) && on(T_G) && t.s != g_ready) {   // the G super-tile must be complete
#ifdef OPD_TRACE
                    const long long w0 = clock64();
#endif
                    wait_counter(bp.g_done + t.s, CG * t.ng);                             // before TMA reads it (checked once
                    fence_proxy_async_all();                                              // per super-tile, not per tile)
                    g_ready = t.s;
#ifdef OPD_TRACE
                    tr[3] += clock64() - w0;
#endif
                }
#ifdef OPD_TRACE
                produce_tile<CG, ST>(P, op, it, [&] { have_next = fetch(nxt); }, tr);
                tr[0] += 1; tr[1] += clock64() - t0;
#else
                produce_tile<CG, ST>(P, op, it, [&] { have_next = fetch(nxt); });
#endif
                t = nxt; have = have_next;
            }
#ifdef OPD_TRACE
            if (bp.trace) {
                for (int ty = 0; ty < 4; ++ty) for (int k = 0; k < 8; ++k)
                    if (trp[ty][k]) atomicAdd(bp.trace + (1 * 4 + ty) * 8 + k, (unsigned long long)trp[ty][k]);
                atomicAdd(bp.trace + 96 + 1, (unsigned long long)(clock64() - k0));
                atomicAdd(bp.trace + 104, (unsigned long long)q_wait); atomicAdd(bp.trace + 105, (unsigned long long)q_copy);
                atomicAdd(bp.trace + 106, (unsigned long long)q_arrive);
            }
#endif
        }
    } else if (warp == 1) {
        // =========================== tile claimer (peer CTA of a pair; this warp has no other work there) =========
        if (CG == 2 && rank == 1 && elect_one()) {
            BwdSched<CG, DENSE> sc; sc.init(bp);
            BwdTile t;
            int n = 0;
            while (claim_next(sc, n, t)) {}
        }
        // =========================== MMA issuer ===========================
        if (rank == 0 && elect_one()) {
            BwdTile t, nxt;
            int it = 0, lt = 0, n = 0;
            auto fetch = [&](BwdTile& o) -> bool { return read_next(n, o); };
#ifdef OPD_TRACE
            long long trm[4][8] = {};
            const long long k0 = clock64();
#endif
            bool have = fetch(t), have_next = false;
            while (have) {
#ifdef OPD_TRACE
                long long* tr = trm[t.type];
                const long long t0 = clock64();
#endif
                int a_mn, b_mn, K;
                if (t.type == T_G) { a_mn = 0; b_mn = (bp.wl == 0); K = bp.d; }
                else if (DENSE && t.type == T_Q) { a_mn = 0; b_mn = (bp.wl_t == 0); K = bp.dT; }
                else if (t.type == T_DX) { a_mn = 0; b_mn = (bp.wl == 1); K = t.Vb_eff; }
                else { a_mn = 1; b_mn = 1; K = t.Tb_eff; }
                // the next tile is read once this tile's first MMAs are queued, not between two tiles
#ifdef OPD_TRACE
                mma_tile<CG, ST>(P, a_mn, b_mn, ((K + BK - 1) / BK) * nseg, lt, it, [&] { have_next = fetch(nxt); }, tr);
                tr[0] += 1; tr[1] += clock64() - t0; tr[6] += ((K + BK - 1) / BK) * nseg;
#else
                mma_tile<CG, ST>(P, a_mn, b_mn, ((K + BK - 1) / BK) * nseg, lt, it, [&] { have_next = fetch(nxt); });
#endif
                ++lt;
                t = nxt; have = have_next;
            }
#ifdef OPD_TRACE
            if (bp.trace) {
                for (int ty = 0; ty < 4; ++ty) for (int k = 0; k < 8; ++k)
                    if (trm[ty][k]) atomicAdd(bp.trace + (0 * 4 + ty) * 8 + k, (unsigned long long)trm[ty][k]);
                atomicAdd(bp.trace + 96 + 0, (unsigned long long)(clock64() - k0));
                atomicAdd(bp.trace + 100, (unsigned long long)q_wait); atomicAdd(bp.trace + 101, (unsigned long long)q_copy);
                atomicAdd(bp.trace + 102, (unsigned long long)q_arrive);
            }
#endif
        }
    } else if (warp < 2 + BWD_EPI_WARPS) {
        // =========================== epilogue warps ===========================
        // Two warps per TMEM lane quarter (warps w and w + 4 share a scheduler): half 0 takes columns 0-127 of a G tile and
        // all of a Q / grad_hidden / grad_W tile (long main loops, staged through this half's shared-memory buffers), half 1
        // columns 128-255 of a G tile.  Both halves follow every tile (queue slot, accumulator stage, publication).
        const int quarter = warp & 3;
        const int half = (warp - 2) >> 2;
        const int row_in_tile = quarter * 32 + lane;
        const int epi_tid = ((warp - 2) & 3) * 32 + lane;
        BwdTile t;
        int lt = 0;
        int c_ready = -1, dx_ready = -1, dw_ready = -1, gq_ready = -1, q_ready = -1;   // dependencies already seen complete (warp-uniform)
#ifdef OPD_TRACE
        long long tre[4][8] = {};
        long long* tr = tre[0];
        const long long k0 = clock64();
#endif
        auto wait_for = [&](const int* counter, int expected) {      // warp-level acquire of a dependency counter
#ifdef OPD_TRACE
            const long long w0 = clock64();
#endif
            if (lane == 0) { wait_counter(counter, expected); fence_proxy_async_all(); }
            __syncwarp();
#ifdef OPD_TRACE
            tr[2] += clock64() - w0;
#endif
        };
        auto acquire = [&]() -> uint32_t {
#ifdef OPD_TRACE
            const long long w0 = clock64();
            const uint32_t ta = epi_acquire<CG, ST>(P, lt, quarter);
            tr[3] += clock64() - w0;
            return ta;
#else
            return epi_acquire<CG, ST>(P, lt, quarter);
#endif
        };
        // Publication of a finished tile (its dependency counter + 1, with release semantics at gpu scope) is the publisher
        // warp's job: the fence it needs waits for the SM's outstanding stores (2000-5000 cycles per tile when the epilogue
        // warps executed it, profiles/r02_trace.md), which the epilogue warps now spend on their next tile.  Each epilogue
        // warp arrives on pub_full once its own stores are issued (per-thread stores; ordered before the arrive's release by
        // the __syncwarp) or complete (TMA stores / reductions: all issued by lane 0, which waits for its bulk groups first).
        // An epilogue warp is never more than two tiles ahead of another one (they meet at the TMEM stage hand-back: every
        // warp waits for every tile's accumulator), so PUB_Q = 4 slots cannot mix arrivals of different rounds; warp 2 waits
        // for the slot itself before it writes the pointer.
        int pn = 0;
        auto hand_over = [&](int* counter) {
            __syncwarp();
            if (lane == 0) {
                bulk_wait<0>();
                if (warp == 2) {
                    mbar_wait(&P.pub_empty[pn % PUB_Q], ((pn / PUB_Q) & 1) ^ 1);
                    *const_cast<int* volatile*>(P.pub_ptr + pn % PUB_Q) = counter;
                }
                mbar_arrive(&P.pub_full[pn % PUB_Q]);
            }
            ++pn;
        };
        for (int n = 0;; ++n) {
#ifdef OPD_TRACE
            const long long t0 = clock64();
#endif
            // each epilogue warp is one reader of the tile queue: lane 0 waits, every lane copies, lane 0 hands the slot back
            if (lane == 0) tile_wait<CG, ST>(P, n);
            __syncwarp();
            tile_copy<CG, ST>(P, n, reinterpret_cast<uint32_t(&)[SCHED_WORDS]>(t));
            __syncwarp();
            if (lane == 0) tile_consumed<CG, ST>(P, n);
            if (!t.valid) { hand_over(nullptr); break; }
#ifdef OPD_TRACE
            tr = tre[t.type];
            tr[5] += clock64() - t0;          // queue wait + copy
#endif
            const int m_blk = t.m_blk * CG + rank;    // this CTA's 128-row block inside the GEMM
            GemmParams gp{};                      // the fields the epilogues read
            gp.tok_off = t.tb0;
#ifdef OPD_TRACE
            gp.tr = tr;
#endif
            // wait for the previous writer / readers of what this epilogue is about to write (and, dense, for its Q tile)
            // (each dependency is checked once per super-tile, not once per tile: a CTA's tiles come in list order)
            const bool works = !(half == 1 && (DENSE || t.type != T_G));      // this warp has columns of the tile to process
            if (!works) {
            } else if (t.type == T_Q) {
                if (t.dep_cnt > 0 && t.s - 2 != gq_ready) { wait_for(bp.g_done + t.s - 2, t.dep_cnt); gq_ready = t.s - 2; }
            } else if (t.type == T_G) {
                const int dep = t.s - bp.gbufs;
                if (t.dep_cnt > 0 && dep > c_ready) {
                    wait_for(bp.dx_done + dep, t.dep_cnt & 0xffff); wait_for(bp.dw_done + dep, t.dep_cnt >> 16); c_ready = dep;
                }
                if (DENSE && on(T_Q) && t.s != q_ready) { wait_for(bp.q_done + t.s, CG * t.ng); q_ready = t.s; }
            } else if (t.type == T_DX) {
                if (t.dep_cnt > 0 && t.s - 1 > dx_ready) { wait_for(bp.dx_done + t.s - 1, t.dep_cnt); dx_ready = t.s - 1; }
            } else {
                if (t.dep_cnt > 0 && t.s - bp.nvb > dw_ready) { wait_for(bp.dw_done + t.s - bp.nvb, t.dep_cnt); dw_ready = t.s - bp.nvb; }
            }
            if (!works) {
                (void)acquire();                                    // nothing to do for this tile: stay in step with the stage
            } else if (DENSE && t.type == T_Q) {
                gp.b_off = t.vb0; gp.N = t.Vb_eff;
                QEpi::Params ep = bp.q;
                ep.qs = static_cast<uint8_t*>(ep.qs) + static_cast<size_t>(t.s & 1) * bp.q_buf_bytes;
                QEpi::State st = QEpi::prepare(ep, gp, m_blk, t.n_blk, row_in_tile, t.Tb_eff);
                const uint32_t taddr = acquire();
                QEpi::run(ep, gp, st, taddr, m_blk, t.n_blk, row_in_tile, t.Tb_eff, nullptr, epi_tid);
            } else if (DENSE && t.type == T_G) {
                gp.b_off = t.vb0; gp.N = t.Vb_eff;
                GDenseEpi::Params ep = bp.gd;
                ep.gs += static_cast<size_t>(t.s % bp.gbufs) * bp.planes * ep.plane_stride;
                ep.qs = static_cast<const uint8_t*>(ep.qs) + static_cast<size_t>(t.s & 1) * bp.q_buf_bytes;
                if (!on(T_DX)) ep.rows = 0;                     // forward-only: nothing consumes G
                GDenseEpi::State st = GDenseEpi::prepare(ep, gp, m_blk, t.n_blk, row_in_tile, t.Tb_eff);
                const uint32_t taddr = acquire();
                GDenseEpi::run(ep, gp, st, taddr, m_blk, t.n_blk, row_in_tile, t.Tb_eff, nullptr, epi_tid);
            } else if (t.type == T_G) {
                gp.b_off = t.vb0; gp.N = t.Vb_eff; gp.row_off = t.s % bp.gbufs;      // ring buffer of this super-tile
                gp.col_off = half * (BN / 2);                                            // this warp's half of the tile's columns
                gp.N = BWD_EPI_WARPS == 8 ? BN / 2 : BN;                                 // tile columns this warp handles
                GEpi::State st = GEpi::prepare(bp.g, gp, m_blk, t.n_blk, row_in_tile, t.Tb_eff);
                const uint32_t taddr = acquire();
                GEpi::run(bp.g, gp, st, taddr, m_blk, t.n_blk, row_in_tile, t.Tb_eff, P.epi_smem, epi_tid);
            } else if (t.type == T_DX) {
                gp.N = bp.d; gp.first = (t.vi == 0); gp.last = (t.vi == bp.nvb - 1);
                DxEpi::State st = DxEpi::prepare(bp.dx, gp, m_blk, t.n_blk, row_in_tile, t.Tb_eff);
                const uint32_t taddr = acquire();
                DxEpi::run(bp.dx, gp, st, taddr, m_blk, t.n_blk, row_in_tile, t.Tb_eff, P.epi_smem, epi_tid);
            } else {
                int M_eff;
                if (bp.wl == 0) { gp.N = t.Vb_eff; gp.row_off = 0; gp.col_off = t.vb0; M_eff = bp.d; }
                else { gp.N = bp.d; gp.row_off = t.vb0; gp.col_off = 0; M_eff = t.Vb_eff; }
                gp.first = bp.dw_store_first && t.tb0 == 0;          // first token super-tile: plain stores
                const uint32_t taddr = acquire();
                DwEpi::run(bp.dw, gp, NoState{}, taddr, m_blk, t.n_blk, row_in_tile, M_eff, P.epi_smem, epi_tid);
            }
            epi_release<CG, ST>(P, lt, lane);                       // TMEM stage free for the MMA warp
            ++lt;
#ifdef OPD_TRACE
            const long long p0 = clock64();
#endif
            // hand the tile to the publisher warp: this warp's stores are issued (generic) or complete (TMA)
            hand_over((t.type == T_G ? bp.g_done : (t.type == T_Q ? bp.q_done : (t.type == T_DX ? bp.dx_done : bp.dw_done))) + t.s);
#ifdef OPD_TRACE
            tr[0] += 1; tr[1] += clock64() - t0; tr[4] += clock64() - p0;
#endif
        }
#ifdef OPD_TRACE
        if (bp.trace && warp == 2 && lane == 0) {
            for (int ty = 0; ty < 4; ++ty) for (int k = 0; k < 8; ++k)
                if (tre[ty][k]) atomicAdd(bp.trace + (2 * 4 + ty) * 8 + k, (unsigned long long)tre[ty][k]);
            atomicAdd(bp.trace + 96 + 2, (unsigned long long)(clock64() - k0));
        }
#endif
    } else {
        // =========================== publisher (last warp) ===========================
        // One thread per CTA: when the four epilogue warps are done with a tile, make their stores visible at gpu scope
        // (the generic-proxy stores of the SM it has observed through the barrier, and the completed bulk stores /
        // reductions) and count the tile on its dependency counter.  Counters count CTA-level epilogues.
        if (lane == 0) {
            for (int n = 0;; ++n) {
                mbar_wait(&P.pub_full[n % PUB_Q], (n / PUB_Q) & 1);
                int* counter = *const_cast<int* volatile*>(P.pub_ptr + n % PUB_Q);
                mbar_arrive(&P.pub_empty[n % PUB_Q]);
                if (counter == nullptr) break;
                fence_proxy_async_all();
                __threadfence();
                atomicAdd(counter, 1);
            }
        }
    }
    P.teardown(warp);
}

}  // namespace opd
