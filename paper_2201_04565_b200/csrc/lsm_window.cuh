// lsm_window.cuh -- the streamed step kernel with WINDOWED neighbour gathers (plain time steps of the product path).
//
// k_gather_stream gathers neighbour positions from global memory (L1 / L2 hits): its warps then sit on the long
// scoreboard for an L2 round trip per tile (ncu, 4096^2 lattice: 5.1 of 11 stall cycles per issue).  With a banded
// numbering the neighbours of a tile of 256 consecutive particles are a handful of short contiguous id ranges (a lattice:
// the tile's own row segment and the segments above and below it; <= 4 ranges, <= 800 particles on every BASELINE.json
// configuration).  Here the producer warp brings those ranges -- the tile's WINDOW -- into the pipeline stage with one
// bulk async copy each, next to the tile's velocities and rows, and the consumers gather from shared memory with a
// 16-bit window index per slot (streamed instead of the 16-bit neighbour offset: same bytes).  No gather leaves the SM,
// no LDG is issued, nothing waits on L2.  Arithmetic, order and breakage handling are those of row_chunk / row_careful
// (slot_eval, particle_math), so exact mode stays bit-identical to the serial reference.
#pragma once
#include "lsm_resident.cuh"

namespace lsmk {

constexpr int kWinMaxSeg = 4;          // contiguous id ranges per tile window

struct __align__(16) TileWin {         // 32 bytes per tile, read by the producer lane only
    int32_t start[kWinMaxSeg];         // first particle of each range
    uint16_t len[kWinMaxSeg];          // particles in each range (0 = unused); ranges are laid out back to back in the stage
    uint16_t own_base;                 // window index of the tile's first own particle
    uint16_t pad[3];
};
static_assert(sizeof(TileWin) == 32, "TileWin must be 32 bytes");

struct WinParams {
    const TileWin *win;                // [T]
    uint16_t *widx;                    // [E] window index of every slot's neighbour (own index for padding / dead slots)
    int win_off;                       // byte offset of the window inside a stage (replaces the own-position block)
};

// The careful pass (see row_careful) over a windowed row: same order, same arithmetic, exact decisions.
template <int PM, bool EXACT>
__device__ __forceinline__ void row_careful_w(const StepParams &P, const WinParams &W, long long step, const RowSrc &R, const double *s_tab, uint32_t win_s,
                                              int p, unsigned own_idx, unsigned w, double2 xp, double &fx, double &fy) {
    fx = 0.0; fy = 0.0;
#pragma unroll 1
    for (unsigned s = 0; s < w; ++s) {
        const unsigned so = s * kSlice;
        const double2 xq = lds_d2(win_s + (uint32_t)reinterpret_cast<const uint16_t *>(R.nbr16)[so] * 16u);
        double k, r0, kr0, dx, dy, r2, g, ue;
        uint32_t thr;
        bool near;
        slot_params<PM>(P, R, s_tab, so, k, r0, kr0, thr);
        slot_eval<EXACT, false>(xq, xp, false, k, r0, kr0, thr, dx, dy, r2, g, ue, near);
        if (near) {
            const size_t e = R.e0 + so;
            double rc;
            if (PM == PM_UNIFORM) rc = P.sp.rc_u;
            else if (PM == PM_TYPED) rc = s_tab[kTabStride * R.typ[so] + 4];
            else rc = __ldg(P.sp.rcS + __ldg(P.sid + e));
            if (__dsqrt_rn(r2) > rc) {   // strict '>' (Q1)
                const int nb = P.nbr[e];                      // the master list names the partner
                P.nbr[e] = p;                                 // dead from now on: every copy of the slot points at its own particle
                P.nbr16[e] = 0;
                W.widx[e] = (uint16_t)own_idx;
                reinterpret_cast<uint16_t *>(const_cast<int16_t *>(R.nbr16))[so] = (uint16_t)own_idx;   // and the staged copy
                if (p < nb) {
                    P.break_step[P.sid[e]] = step;
                    atomicAdd(P.nbroken + spec_of(P.poff, P.B, p), 1ULL);
                }
                continue;
            }
        }
        fx = mad<EXACT>(g, dx, fx);
        fy = mad<EXACT>(g, dy, fy);
    }
}

// CH springs of a windowed row: row_chunk_s with absolute 16-bit window indices instead of signed offsets.
template <int PM, bool EXACT, int CH>
__device__ __forceinline__ bool row_chunk_w(const StepParams &P, const RowS &A, uint32_t tab_s, uint32_t win_s, double2 xp, double &fx, double &fy) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    constexpr bool kHasThr = (PM == PM_RCF || PM == PM_KRT_RCF || PM == PM_FULL);
    uint32_t nb[CH];
    double2 xq[CH];
    bool any_near = false;
    static_for<CH>([&](auto ic) { constexpr int C = decltype(ic)::value; nb[C] = lds_u16o<C * kSlice * 2>(A.nbr); });
#pragma unroll
    for (int c = 0; c < CH; ++c) xq[c] = lds_d2(win_s + nb[c] * 16u);
    static_for<CH>([&](auto ic) {
        constexpr int C = decltype(ic)::value;
        double k, r0 = 0.0, kr0, dx, dy, r2, g, ue;
        uint32_t thr;
        bool near;
        if constexpr (kTab) {
            const uint32_t ta = tab_s + lds_u8o<C * kSlice>(A.typ) * (uint32_t)(kTabStride * 8);
            const double2 kk = lds_d2(ta);
            k = kk.x; kr0 = kk.y;
            if (EXACT) r0 = lds_f64o<24>(ta);
            thr = PM == PM_TYPED ? lds_u32o<16>(ta) : P.sp.thr_base + lds_u8o<C * kSlice * kThrB>(A.thr) * P.sp.thr_mul;
        } else if constexpr (PM == PM_FULL) {
            k = lds_f64o<C * kSlice * 8>(A.kF); r0 = lds_f64o<C * kSlice * 8>(A.r0F); kr0 = k * r0;
            thr = P.sp.thr_base + lds_u8o<C * kSlice * kThrB>(A.thr) * P.sp.thr_mul;
        } else {
            k = P.sp.k_u; r0 = P.sp.r0_u; kr0 = P.sp.kr0_u;
            thr = kHasThr ? P.sp.thr_base + lds_u8o<C * kSlice * kThrB>(A.thr) * P.sp.thr_mul : P.sp.thr_u;
        }
        slot_eval<EXACT, false>(xq[C], xp, false, k, r0, kr0, thr, dx, dy, r2, g, ue, near);
        fx = mad<EXACT>(g, dx, fx);
        fy = mad<EXACT>(g, dy, fy);
        any_near |= near;
    });
    return any_near;
}

// One plain time step (force -> damping + kick2 -> kick1 + drift), persistent CTAs, warp 8 = producer.
template <int PM, bool EXACT>
__global__ void __launch_bounds__(kTile + 32, kStreamMinB) k_gather_win(const StepParams P, const StageLayout L, const WinParams W) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    constexpr bool kHasThr = (PM == PM_RCF || PM == PM_KRT_RCF || PM == PM_FULL);
    constexpr bool kHasKR = (PM == PM_FULL);
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);          // [kMaxStages]
    uint64_t *empty = full + kMaxStages;                            // [kMaxStages]
    double *s_tab = reinterpret_cast<double *>(smem + kStreamHdrBytes);
    unsigned char *stage0 = smem + L.first;
    const int tid = threadIdx.x, wi = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < L.stages; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, kTileSlices); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (kTab) for (int i = tid; i < kTabStride * P.sp.ntypes; i += kTile + 32) s_tab[i] = P.sp.tab[i];
    __syncthreads();

    if (wi == kTileSlices) {  // ---------------- producer warp ----------------
        if (lane == 0) {
            int s = 0; unsigned u = 0;
            uint32_t o0n = 0, o8n = 0;
            int4 wa = make_int4(0, 0, 0, 0), wb = make_int4(0, 0, 0, 0);      // the next tile's TileWin
            if ((long long)blockIdx.x < P.T) {
                o0n = __ldg(&P.hdr[blockIdx.x].off[0]); o8n = __ldg(&P.hdr[blockIdx.x].off[kTileSlices]);
                const int4 *q = reinterpret_cast<const int4 *>(W.win + blockIdx.x);
                wa = __ldg(q); wb = __ldg(q + 1);
            }
            for (long long t = blockIdx.x; t < P.T; t += gridDim.x) {
                const TileHdr *h = P.hdr + t;
                const uint32_t o0 = o0n, ns = o8n - o0n;
                const int st[kWinMaxSeg] = {wa.x, wa.y, wa.z, wa.w};
                const unsigned ln[kWinMaxSeg] = {(unsigned)wb.x & 0xFFFFu, (unsigned)wb.x >> 16, (unsigned)wb.y & 0xFFFFu, (unsigned)wb.y >> 16};
                if (t + gridDim.x < P.T) {   // the next tile's extents and window, ahead of the wait
                    o0n = __ldg(&h[gridDim.x].off[0]); o8n = __ldg(&h[gridDim.x].off[kTileSlices]);
                    const int4 *q = reinterpret_cast<const int4 *>(W.win + t + gridDim.x);
                    wa = __ldg(q); wb = __ldg(q + 1);
                }
                if (u > 0) mbar_wait(empty + s, (u - 1) & 1);
                const unsigned nwin = ln[0] + ln[1] + ln[2] + ln[3];
                unsigned bytes = nwin * 16 + kTile * 16 + kTile + 64 + ns * (kSlice * 2);
                if (kHasThr) bytes += ns * (kSlice * kThrB);
                if (kTab) bytes += ns * kSlice;
                if (kHasKR) bytes += 2 * ns * (kSlice * 8);
                unsigned char *b = stage0 + (size_t)s * L.bytes;
                mbar_expect_tx(full + s, bytes);
                unsigned woff = 0;
#pragma unroll
                for (int q = 0; q < kWinMaxSeg; ++q)
                    if (ln[q]) { bulk_g2s(b + L.pos + woff * 16, P.pos_cur + st[q], ln[q] * 16, full + s); woff += ln[q]; }
                bulk_g2s(b + L.vel, reinterpret_cast<const char *>(P.vel) + t * (kTile * 16), kTile * 16, full + s);
                bulk_g2s(b + L.grp, P.grp + t * kTile, kTile, full + s);
                bulk_g2s(b + L.hdr, h, 64, full + s);
                if (ns) {
                    const size_t e = (size_t)o0 * kSlice;
                    bulk_g2s(b + L.nbr, W.widx + e, ns * (kSlice * 2), full + s);
                    if (kHasThr) bulk_g2s(b + L.thr, P.sp.thr + e, ns * (kSlice * kThrB), full + s);
                    if (kTab) bulk_g2s(b + L.typ, P.sp.typ + e, ns * kSlice, full + s);
                    if (kHasKR) {
                        bulk_g2s(b + L.kF, P.sp.kF + e, ns * (kSlice * 8), full + s);
                        bulk_g2s(b + L.r0F, P.sp.r0F + e, ns * (kSlice * 8), full + s);
                    }
                }
                if (++s == L.stages) { s = 0; ++u; }
            }
        }
        return;
    }
    // ---------------- consumer warps: thread = particle ----------------
    const uint32_t stage_s0 = smem_u32(stage0), tab_s = smem_u32(s_tab);
    const StepVar V{P.pos_cur, P.pos_next, P.step, 0u};
    int s = 0; unsigned u = 0;
    for (long long t = blockIdx.x; t < P.T; t += gridDim.x) {
        mbar_wait(full + s, u & 1);
        const uint32_t b_s = stage_s0 + (uint32_t)s * (uint32_t)L.bytes;
        const long long p = t * kTile + tid;
        if (p < P.N) {
            const uint32_t hdr_s = b_s + (uint32_t)L.hdr;
            const unsigned w = lds_u8(hdr_s + 36u + (uint32_t)wi);                       // TileHdr: off[9], w[8], own_base
            const uint32_t off_w = lds_u32o<0>(hdr_s + (uint32_t)wi * 4u), off_0 = lds_u32o<0>(hdr_s);
            const unsigned own_idx = (lds_u32o<44>(hdr_s) & 0xFFFFu) + (unsigned)tid;
            const unsigned rel = (off_w - off_0) * kSlice + lane;
            const uint32_t win_s = b_s + (uint32_t)L.pos;
            const double2 xp = lds_d2(win_s + own_idx * 16u);
            const double2 vh = lds_d2(b_s + (uint32_t)L.vel + (uint32_t)tid * 16u);
            const uint8_t g = (uint8_t)lds_u8(b_s + (uint32_t)L.grp + (uint32_t)tid);
            RowS A;
            A.nbr = b_s + (uint32_t)L.nbr + rel * 2; A.thr = b_s + (uint32_t)L.thr + rel * kThrB; A.typ = b_s + (uint32_t)L.typ + rel;
            A.kF = b_s + (uint32_t)L.kF + rel * 8; A.r0F = b_s + (uint32_t)L.r0F + rel * 8;
            double fx = 0.0, fy = 0.0;
            bool any_near = false;
            constexpr int CH = kRowCH;
            unsigned s0 = 0;
            for (; s0 + CH <= w; s0 += CH) {
                any_near |= row_chunk_w<PM, EXACT, CH>(P, A, tab_s, win_s, xp, fx, fy);
                A.nbr += CH * kSlice * 2; A.thr += CH * kSlice * kThrB; A.typ += CH * kSlice; A.kF += CH * kSlice * 8; A.r0F += CH * kSlice * 8;
            }
            for (; s0 < w; ++s0) {
                any_near |= row_chunk_w<PM, EXACT, 1>(P, A, tab_s, win_s, xp, fx, fy);
                A.nbr += kSlice * 2; A.thr += kSlice * kThrB; A.typ += kSlice; A.kF += kSlice * 8; A.r0F += kSlice * 8;
            }
            if (any_near) {   // rare: redo the row deciding exactly
                unsigned char *b = stage0 + (size_t)s * L.bytes;
                RowSrc R;
                R.nbr = nullptr;
                R.nbr16 = reinterpret_cast<const int16_t *>(b + L.nbr) + rel;
                R.thr = reinterpret_cast<const thr_t *>(b + L.thr) + rel;
                R.typ = (b + L.typ) + rel;
                R.kF = reinterpret_cast<const double *>(b + L.kF) + rel;
                R.r0F = reinterpret_cast<const double *>(b + L.r0F) + rel;
                R.e0 = (size_t)off_w * kSlice + lane;
                row_careful_w<PM, EXACT>(P, W, P.step, R, s_tab, win_s, (int)p, own_idx, w, xp, fx, fy);
            }
            particle_update<EXACT, true, true, false>(P, V, p, xp, vh, g, fx, fy, 0.0);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + s);
        if (++s == L.stages) { s = 0; ++u; }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Several plain time steps in ONE cooperative launch for L2-resident lattices, with windows (k_coop_win).
// Every CTA keeps its tiles' rows, velocities and group bytes in its pipeline stages for the whole launch (as the resident
// mode of k_gather_stream<MULTI> does) and re-fetches only the position WINDOW of each tile per step, by bulk async copy
// from the position buffer all CTAs have just written -- after the same grid barrier (one global arrival counter).  The
// consumers then gather from shared memory instead of paying an L2 round trip per tile behind the barrier.
// ---------------------------------------------------------------------------------------------------------------
struct CoopWinParams {
    const TileWin *win;
    uint16_t *widx;
    unsigned long long *gbar;          // global arrival counter (monotonic across launches)
    unsigned long long gbar_base;      // its value before this launch
    double2 *pos_a, *pos_b;            // step i reads pos_a / writes pos_b when i is even, the reverse when odd
    int nsteps;
};

template <int PM, bool EXACT>
__global__ void __launch_bounds__(kTile + 32, kStreamMinB) k_coop_win(const StepParams P, const StageLayout L, const CoopWinParams Q) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    constexpr bool kHasThr = (PM == PM_RCF || PM == PM_KRT_RCF || PM == PM_FULL);
    constexpr bool kHasKR = (PM == PM_FULL);
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);          // [kMaxStages] window (and, first, whole tile) landed
    uint64_t *stepdone = full + 2 * kMaxStages;                    // all consumer warps finished the step
    double *s_tab = reinterpret_cast<double *>(smem + kStreamHdrBytes);
    unsigned char *stage0 = smem + L.first;
    const int tid = threadIdx.x, wi = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < L.stages; ++s) mbar_init(full + s, 1);
        mbar_init(stepdone, kTileSlices);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (kTab) for (int i = tid; i < kTabStride * P.sp.ntypes; i += kTile + 32) s_tab[i] = P.sp.tab[i];
    __syncthreads();
    const WinParams W{Q.win, Q.widx, L.pos};

    if (wi == kTileSlices) {  // ---------------- producer warp ----------------
        for (int it = 0; it < Q.nsteps; ++it) {
            const double2 *pos_cur = (it & 1) ? Q.pos_b : Q.pos_a;
            if (it > 0 && lane == 0) {   // grid barrier: every CTA has finished (and published) step it - 1
                mbar_wait(stepdone, (unsigned)(it - 1) & 1u);
                grid_arrive_and_wait(Q.gbar, Q.gbar_base + (unsigned long long)it * gridDim.x);
                asm volatile("fence.proxy.async;" ::: "memory");          // their generic-proxy stores before our bulk copies
            }
            if (lane == 0) {
                int s = 0;
                for (long long t = blockIdx.x; t < P.T; t += gridDim.x, ++s) {
                    const TileWin tw = Q.win[t];
                    unsigned nwin = 0;
#pragma unroll
                    for (int q = 0; q < kWinMaxSeg; ++q) nwin += tw.len[q];
                    unsigned char *b = stage0 + (size_t)s * L.bytes;
                    unsigned bytes = nwin * 16;
                    const TileHdr *h = P.hdr + t;
                    const uint32_t o0 = h->off[0], ns = h->off[kTileSlices] - h->off[0];
                    if (it == 0) {
                        bytes += kTile * 16 + kTile + 64 + ns * (kSlice * 2);
                        if (kHasThr) bytes += ns * (kSlice * kThrB);
                        if (kTab) bytes += ns * kSlice;
                        if (kHasKR) bytes += 2 * ns * (kSlice * 8);
                    }
                    mbar_expect_tx(full + s, bytes);
                    unsigned woff = 0;
#pragma unroll
                    for (int q = 0; q < kWinMaxSeg; ++q)
                        if (tw.len[q]) { bulk_g2s(b + L.pos + woff * 16, pos_cur + tw.start[q], tw.len[q] * 16u, full + s); woff += tw.len[q]; }
                    if (it == 0) {   // rows, velocities and group bytes stay for the whole launch
                        bulk_g2s(b + L.vel, reinterpret_cast<const char *>(P.vel) + t * (kTile * 16), kTile * 16, full + s);
                        bulk_g2s(b + L.grp, P.grp + t * kTile, kTile, full + s);
                        bulk_g2s(b + L.hdr, h, 64, full + s);
                        if (ns) {
                            const size_t e = (size_t)o0 * kSlice;
                            bulk_g2s(b + L.nbr, Q.widx + e, ns * (kSlice * 2), full + s);
                            if (kHasThr) bulk_g2s(b + L.thr, P.sp.thr + e, ns * (kSlice * kThrB), full + s);
                            if (kTab) bulk_g2s(b + L.typ, P.sp.typ + e, ns * kSlice, full + s);
                            if (kHasKR) {
                                bulk_g2s(b + L.kF, P.sp.kF + e, ns * (kSlice * 8), full + s);
                                bulk_g2s(b + L.r0F, P.sp.r0F + e, ns * (kSlice * 8), full + s);
                            }
                        }
                    }
                }
            }
            __syncwarp();
        }
        return;
    }
    // ---------------- consumer warps: thread = particle ----------------
    const uint32_t stage_s0 = smem_u32(stage0), tab_s = smem_u32(s_tab);
    for (int it = 0; it < Q.nsteps; ++it) {
        StepVar V;
        V.pos_cur = (it & 1) ? Q.pos_b : Q.pos_a; V.pos_next = (it & 1) ? Q.pos_a : Q.pos_b; V.step = P.step + it; V.pos_s = 0u;
        const bool last = it + 1 == Q.nsteps;
        int s = 0;
        for (long long t = blockIdx.x; t < P.T; t += gridDim.x, ++s) {
            mbar_wait(full + s, (unsigned)it & 1u);
            const uint32_t b_s = stage_s0 + (uint32_t)s * (uint32_t)L.bytes;
            const long long p = t * kTile + tid;
            if (p < P.N) {
                const uint32_t hdr_s = b_s + (uint32_t)L.hdr;
                const unsigned w = lds_u8(hdr_s + 36u + (uint32_t)wi);
                const uint32_t off_w = lds_u32o<0>(hdr_s + (uint32_t)wi * 4u), off_0 = lds_u32o<0>(hdr_s);
                const unsigned own_idx = (lds_u32o<44>(hdr_s) & 0xFFFFu) + (unsigned)tid;
                const unsigned rel = (off_w - off_0) * kSlice + lane;
                const uint32_t win_s = b_s + (uint32_t)L.pos;
                const uint32_t vel_a = b_s + (uint32_t)L.vel + (uint32_t)tid * 16u;
                const double2 xp = lds_d2(win_s + own_idx * 16u);
                const double2 vh = lds_d2(vel_a);
                const uint8_t g = (uint8_t)lds_u8(b_s + (uint32_t)L.grp + (uint32_t)tid);
                RowS A;
                A.nbr = b_s + (uint32_t)L.nbr + rel * 2; A.thr = b_s + (uint32_t)L.thr + rel * kThrB; A.typ = b_s + (uint32_t)L.typ + rel;
                A.kF = b_s + (uint32_t)L.kF + rel * 8; A.r0F = b_s + (uint32_t)L.r0F + rel * 8;
                double fx = 0.0, fy = 0.0;
                bool any_near = false;
                constexpr int CH = kRowCH;
                unsigned s0 = 0;
                for (; s0 + CH <= w; s0 += CH) {
                    any_near |= row_chunk_w<PM, EXACT, CH>(P, A, tab_s, win_s, xp, fx, fy);
                    A.nbr += CH * kSlice * 2; A.thr += CH * kSlice * kThrB; A.typ += CH * kSlice; A.kF += CH * kSlice * 8; A.r0F += CH * kSlice * 8;
                }
                for (; s0 < w; ++s0) {
                    any_near |= row_chunk_w<PM, EXACT, 1>(P, A, tab_s, win_s, xp, fx, fy);
                    A.nbr += kSlice * 2; A.thr += kSlice * kThrB; A.typ += kSlice; A.kF += kSlice * 8; A.r0F += kSlice * 8;
                }
                if (any_near) {
                    unsigned char *b = stage0 + (size_t)s * L.bytes;
                    RowSrc R;
                    R.nbr = nullptr;
                    R.nbr16 = reinterpret_cast<const int16_t *>(b + L.nbr) + rel;
                    R.thr = reinterpret_cast<const thr_t *>(b + L.thr) + rel;
                    R.typ = (b + L.typ) + rel;
                    R.kF = reinterpret_cast<const double *>(b + L.kF) + rel;
                    R.r0F = reinterpret_cast<const double *>(b + L.r0F) + rel;
                    R.e0 = (size_t)off_w * kSlice + lane;
                    row_careful_w<PM, EXACT>(P, W, V.step, R, s_tab, win_s, (int)p, own_idx, w, xp, fx, fy);
                }
                const Upd o = particle_math<EXACT, true, true, false>(P, V.step, p, xp, vh, g, fx, fy);
                V.pos_next[p] = o.xn;                                   // the neighbours' (and our own) next windows come from here
                if (g == kFree) { sts_d2(vel_a, o.w); if (last) P.vel[p] = o.w; }
            }
            __syncwarp();
        }
        if (!last) { __syncwarp(); if (lane == 0) mbar_arrive(stepdone); }
    }
}

}  // namespace lsmk
