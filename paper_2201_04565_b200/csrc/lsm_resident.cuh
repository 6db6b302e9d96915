// lsm_resident.cuh -- cluster-resident time stepping ("high-throughput ... data
// generation": many small specimens, or one tiny lattice).
//
// One thread-block cluster owns one UNIT (a specimen of a batch, or a whole small lattice) for a whole run of plain time
// steps: its state is loaded from HBM once, stepped in shared memory, and stored once.  HBM traffic per time step falls
// by the run length, the per-step grid barrier (a global atomic counter all CTAs spin on) becomes a hardware cluster
// barrier, and every neighbour gather becomes a shared-memory load.
//
//   * The unit's slices (32 consecutive particles) are split into contiguous ranges, one per CTA of the cluster.
//   * Each CTA keeps, in shared memory: a WINDOW of positions = its own particles plus the ghosts its rows reference
//     (with a banded numbering -- the condition under which the 16-bit neighbour offsets exist -- that is one contiguous
//     id range), double-buffered; its own half-step velocities and group bytes; its rows of the sliced-ELL lists.
//   * A step reads buffer `cur` and writes buffer `cur ^ 1`.  A particle that is a ghost elsewhere is also written into
//     the other CTA's window through distributed shared memory (st.shared::cluster on a mapa address).
//   * Synchronisation per step is by data flow, not by a barrier: a ghost is pushed with st.async ... mbarrier::complete_tx
//     on the RECEIVING CTA's mbarrier, which that CTA armed with the byte count of all its ghosts; its boundary warps
//     wait for the phase (~100 cycles when the data is there) before they read ghosts, interior warps never wait, and
//     __syncthreads closes the step inside the CTA.  (A release / acquire barrier.cluster per step was measured at
//     340-480 cycles on B200, a relaxed one at 75-140; the transaction barrier needs neither fence.)  Overwriting a
//     ghost slot two steps later is safe because a CTA only receives the pushes of step n + 1 from a neighbour after
//     that neighbour's boundary slices have read the ghosts of step n + 1 -- the spring graph is symmetric, so the
//     slices that push to a CTA are exactly the slices that read its particles.
//   * Row evaluation and the particle update are the functions of lsm_kernels.cuh (row_forces with GM_SMEM gathers,
//     particle_math): the same arithmetic in the same order as the direct and streamed kernels, so exact mode stays
//     bit-identical to the serial reference.  Breakage marks go to the global lists and to the resident copy.
//   * Only plain time steps run here; sample steps, the last step of an lsm_step call and compaction are the streamed
//     kernel's (one launch each), exactly as for the cooperative multi-step launch.
#pragma once
#include "lsm_kernels.cuh"

namespace lsmk {

constexpr int kResThreads = 512;       // 16 warps, one CTA per SM (the window fills most of its shared memory); measured on
                                       // 128 specimens of 128^2: 512 threads 32.6 us per step, 768 34.3, 1024 33.6
constexpr int kResCH = 6;              // springs of a row evaluated together
constexpr int kResMaxPush = 6;         // other CTAs of the cluster a CTA has ghosts in (2 for a banded lattice numbering)
constexpr int kResMaxCluster = 16;     // 8 portable, 16 with cudaFuncAttributeNonPortableClusterSizeAllowed

struct ResPush { int32_t rank, lo, hi, rwlo; };   // own particles [lo, hi) are ghosts of CTA `rank`, whose window starts at rwlo

struct ResCta {                 // one per CTA of a resident launch (built at create)
    int32_t own_lo;             // first own particle (internal id, multiple of 32)
    int32_t n_own;              // own particles (the last slice of the last unit may be ragged)
    int32_t sl0, n_sl;          // first own slice (global slice index), number of own slices
    int32_t wlo, wlen;          // window [wlo, wlo + wlen): own particles and ghosts
    int32_t n_boundary;         // the first n_boundary entries of this CTA's order list are its boundary slices
    int32_t n_push;
    ResPush push[kResMaxPush];
};

struct ResLayout {              // byte offsets inside dynamic shared memory, the same in every CTA of the launch
    int tab, pos0, pos1, vel, grp, sl_off, nbr, thr, typ, kF, r0F;
    int bytes;
    int win_cap, own_cap, sl_cap, slot_cap;   // capacities (particles, particles, slices, slots of 32 entries)
};

struct ResParams {
    const ResCta *desc;         // [grid]
    const uint16_t *order;      // [grid][sl_cap] local slice indices, boundary slices first
    double2 *pos_io;            // positions: read at the start, overwritten with the result (in place)
    int nsteps;
};

__device__ __forceinline__ unsigned cluster_ctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ uint32_t map_to_rank(uint32_t saddr, unsigned rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
// ghost push: the store and the completion of 16 transaction bytes on the receiver's mbarrier travel together
__device__ __forceinline__ void st_async_d2(uint32_t addr, double2 v, uint32_t mbar) {
    asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(addr), "d"(v.x), "d"(v.y), "r"(mbar) : "memory");
}
__device__ __forceinline__ void sts_d2(uint32_t addr, double2 v) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}

template <class T> __device__ __forceinline__ void res_copy16(void *dst, const T *src, size_t bytes, int tid) {   // 16-byte aligned, multiple of 16
    const uint4 *s4 = reinterpret_cast<const uint4 *>(src);
    uint4 *d4 = reinterpret_cast<uint4 *>(dst);
    for (size_t i = tid; i < bytes / 16; i += kResThreads) d4[i] = __ldg(s4 + i);
}

__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }

// CH springs of one row from the resident copy: the arithmetic of row_chunk (slot_eval, same accumulation order), the
// loads spelled as ld.shared [reg + immediate].  pos_p: shared address of the particle's own position in the current buffer.
template <int PM, bool EXACT, int CH>
__device__ __forceinline__ bool row_chunk_s(const StepParams &P, const RowS &A, uint32_t tab_s, uint32_t pos_p, double2 xp, double &fx, double &fy) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    constexpr bool kHasThr = (PM == PM_RCF || PM == PM_KRT_RCF || PM == PM_FULL);
    int nb[CH];
    double2 xq[CH];
    bool any_near = false;
    static_for<CH>([&](auto ic) { constexpr int C = decltype(ic)::value; nb[C] = lds_s16o<C * kSlice * 2>(A.nbr); });
#pragma unroll
    for (int c = 0; c < CH; ++c) xq[c] = lds_d2(pos_p + (uint32_t)(nb[c] * 16));
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

template <int PM, bool EXACT>
__global__ void __launch_bounds__(kResThreads, 1) k_resident(const StepParams P, const ResLayout L, const ResParams Q) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    constexpr bool kHasThr = (PM == PM_RCF || PM == PM_KRT_RCF || PM == PM_FULL);
    constexpr bool kHasKR = (PM == PM_FULL);
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ ResCta d;
    __shared__ __align__(8) uint64_t ghost_bar[2];  // transaction barriers, alternating by step parity: a phase completes when all
                                                    // ghosts of that step are in.  Two of them, so that the barrier a slow warp still has to
                                                    // test cannot run a phase ahead (its next phase is armed only after the step's __syncthreads)
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int nwarps = kResThreads / 32;
    if (tid < (int)(sizeof(ResCta) / 4)) reinterpret_cast<int32_t *>(&d)[tid] = reinterpret_cast<const int32_t *>(Q.desc + blockIdx.x)[tid];
    if (tid == 0) { mbar_init(&ghost_bar[0], 1); mbar_init(&ghost_bar[1], 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
    __syncthreads();
    // the hot loop keeps these in registers (d itself stays in shared memory for the push table)
    const int own_lo = d.own_lo, n_own = d.n_own, sl0 = d.sl0, n_sl = d.n_sl, wlo = d.wlo, wlen = d.wlen, n_boundary = d.n_boundary, n_push = d.n_push;

    double *s_tab = reinterpret_cast<double *>(smem + L.tab);
    double2 *s_vel = reinterpret_cast<double2 *>(smem + L.vel);
    uint8_t *s_grp = smem + L.grp;
    uint2 *s_slice = reinterpret_cast<uint2 *>(smem + L.sl_off);     // per entry of the order list: {slice | width << 16, slot offset}
    const uint32_t posA = smem_u32(smem + L.pos0), posB = smem_u32(smem + L.pos1);
    const uint32_t vel_s = smem_u32(s_vel), grp_s = smem_u32(s_grp), slice_s = smem_u32(s_slice);

    // ---------------- load: window positions, own velocities / groups, slice table, rows ----------------
    uint32_t slot0 = 0;
    if (n_sl > 0) {
        slot0 = __ldg(&P.hdr[sl0 >> 3].off[sl0 & 7]);
        const int sl_end = sl0 + n_sl;                          // end slot = start of the next slice, or the tile's end entry
        const uint32_t slot1 = (sl_end & 7) ? __ldg(&P.hdr[sl_end >> 3].off[sl_end & 7]) : __ldg(&P.hdr[(sl_end >> 3) - 1].off[kTileSlices]);
        const size_t e0 = (size_t)slot0 * kSlice, ne = (size_t)(slot1 - slot0) * kSlice;
        res_copy16(smem + L.nbr, P.nbr16 + e0, ne * 2, tid);
        if (kHasThr) res_copy16(smem + L.thr, P.sp.thr + e0, ne * kThrB, tid);
        if (kTab) res_copy16(smem + L.typ, P.sp.typ + e0, ne, tid);
        if (kHasKR) { res_copy16(smem + L.kF, P.sp.kF + e0, ne * 8, tid); res_copy16(smem + L.r0F, P.sp.r0F + e0, ne * 8, tid); }
    }
    if (kTab) for (int i = tid; i < kTabStride * P.sp.ntypes; i += kResThreads) s_tab[i] = P.sp.tab[i];
    for (int i = tid; i < wlen; i += kResThreads) reinterpret_cast<double2 *>(smem + L.pos0)[i] = Q.pos_io[wlo + i];
    for (int i = tid; i < n_sl * kSlice; i += kResThreads) { s_vel[i] = P.vel[own_lo + i]; s_grp[i] = P.grp[own_lo + i]; }
    for (int i = tid; i < n_sl; i += kResThreads) {             // entry i of the order list (boundary slices first)
        const int ls = Q.order[(size_t)blockIdx.x * L.sl_cap + i], gs = sl0 + ls;
        s_slice[i] = make_uint2((uint32_t)ls | ((uint32_t)P.hdr[gs >> 3].w[gs & 7] << 16), __ldg(&P.hdr[gs >> 3].off[gs & 7]) - slot0);
    }
    __syncthreads();
    cluster_arrive();     // every CTA of the cluster is running and has its window before anyone writes into a neighbour's
    cluster_wait();

    // ---------------- one slice of one step: lane = particle ----------------
    const uint32_t tab_s = smem_u32(s_tab), bar_s = smem_u32(&ghost_bar[0]);
    const unsigned ghost_bytes = (unsigned)(wlen - n_own) * 16u;   // every window particle that is not mine is pushed to me each step
    RowS lane_rows;    // shared addresses of this lane's entry in slot 0 of the CTA's row block
    lane_rows.nbr = smem_u32(smem + L.nbr) + lane * 2; lane_rows.thr = smem_u32(smem + L.thr) + lane * kThrB; lane_rows.typ = smem_u32(smem + L.typ) + lane;
    lane_rows.kF = smem_u32(smem + L.kF) + lane * 8; lane_rows.r0F = smem_u32(smem + L.r0F) + lane * 8;
    auto do_slice = [&](int k, uint32_t pc, uint32_t pn, long long step, bool push, uint32_t push_bar) {
        const uint2 se = lds_u2(slice_s + (uint32_t)k * 8u);
        const int li = (int)(se.x & 0xFFFFu) * kSlice + lane;     // index among own particles
        if (li >= n_own) return;
        const int p = own_lo + li;
        const unsigned w = se.x >> 16;
        const uint32_t pos_p = pc + (uint32_t)(p - wlo) * 16u;
        const double2 xp = lds_d2(pos_p);
        const double2 vh = lds_d2(vel_s + (uint32_t)li * 16u);
        const uint8_t g = (uint8_t)lds_u8(grp_s + (uint32_t)li);
        RowS A;
        A.nbr = lane_rows.nbr + se.y * (kSlice * 2); A.thr = lane_rows.thr + se.y * (kSlice * kThrB); A.typ = lane_rows.typ + se.y * kSlice;
        A.kF = lane_rows.kF + se.y * (kSlice * 8); A.r0F = lane_rows.r0F + se.y * (kSlice * 8);
        double fx = 0.0, fy = 0.0;
        bool any_near = false;
        constexpr int CH = kResCH;
        unsigned s0 = 0;
        for (; s0 + CH <= w; s0 += CH) {
            any_near |= row_chunk_s<PM, EXACT, CH>(P, A, tab_s, pos_p, xp, fx, fy);
            A.nbr += CH * kSlice * 2; A.thr += CH * kSlice * kThrB; A.typ += CH * kSlice; A.kF += CH * kSlice * 8; A.r0F += CH * kSlice * 8;
        }
        for (; s0 < w; ++s0) {
            any_near |= row_chunk_s<PM, EXACT, 1>(P, A, tab_s, pos_p, xp, fx, fy);
            A.nbr += kSlice * 2; A.thr += kSlice * kThrB; A.typ += kSlice; A.kF += kSlice * 8; A.r0F += kSlice * 8;
        }
        if (any_near) {   // rare: a spring came close to its breaking length -> redo the row deciding exactly (row_careful)
            const unsigned rel = se.y * kSlice + lane;
            RowSrc R;
            R.nbr = nullptr;
            R.nbr16 = reinterpret_cast<const int16_t *>(smem + L.nbr) + rel;
            R.thr = reinterpret_cast<const thr_t *>(smem + L.thr) + rel;
            R.typ = (smem + L.typ) + rel;
            R.kF = reinterpret_cast<const double *>(smem + L.kF) + rel;
            R.r0F = reinterpret_cast<const double *>(smem + L.r0F) + rel;
            R.e0 = (size_t)(slot0 + se.y) * kSlice + lane;
            StepVar V;
            V.pos_cur = nullptr; V.pos_next = nullptr; V.step = step;
            V.pos_s = pc - (uint32_t)wlo * 16u;
            double uu = 0.0;
            row_careful<PM, EXACT, false, GM_SMEM, true>(P, V, R, s_tab, p, w, xp, fx, fy, uu);
        }
        const Upd o = particle_math<EXACT, true, true, false>(P, step, p, xp, vh, g, fx, fy);
        sts_d2(pn + (uint32_t)(p - wlo) * 16u, o.xn);
        if (g == kFree) sts_d2(vel_s + (uint32_t)li * 16u, o.w);
        if (push) {
            for (int q = 0; q < n_push; ++q)
                if (p >= d.push[q].lo && p < d.push[q].hi)
                    st_async_d2(map_to_rank(pn + (uint32_t)(p - d.push[q].rwlo) * 16u, (unsigned)d.push[q].rank), o.xn,
                                map_to_rank(push_bar, (unsigned)d.push[q].rank));
        }
    };

    // ---------------- time steps ----------------
    // Warp w takes entries w, w + 16, ... of the order list: its boundary slices first (they need this step's ghosts and
    // push the next step's), then its interior ones -- every warp gets the same number of slices (+-1).
    bool cur = false;
    for (int it = 0; it < Q.nsteps; ++it) {
        const bool more = it + 1 < Q.nsteps;
        const uint32_t pc = cur ? posB : posA, pn = cur ? posA : posB;
        int k = warp;
        if (k < n_boundary) {
            if (it > 0) mbar_wait(&ghost_bar[(it - 1) & 1], (unsigned)((it - 1) >> 1) & 1u);   // the ghosts pushed during step it - 1 are in
            if (tid == 0 && more) mbar_expect_tx(&ghost_bar[it & 1], ghost_bytes);              // arm the phase that collects this step's pushes
            for (; k < n_boundary; k += nwarps) do_slice(k, pc, pn, P.step + it, more, bar_s + (uint32_t)(it & 1) * 8u);
        }
        for (; k < n_sl; k += nwarps) do_slice(k, pc, pn, P.step + it, false, 0u);
        __syncthreads();                                       // own-region writes of this step before anyone's next step
        cur = !cur;
    }
    cluster_arrive_relaxed();                                  // no CTA leaves while a neighbour may still be pushing into it
    cluster_wait();

    // ---------------- store the own particles ----------------
    const double2 *res = reinterpret_cast<const double2 *>(smem + (cur ? L.pos1 : L.pos0)) + (own_lo - wlo);
    for (int i = tid; i < n_own; i += kResThreads) { Q.pos_io[own_lo + i] = res[i]; P.vel[own_lo + i] = s_vel[i]; }
}

}  // namespace lsmk
