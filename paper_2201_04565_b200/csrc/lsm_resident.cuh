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
//   * Synchronisation per step: barrier.cluster.arrive (release) after the BOUNDARY slices (those exchanging ghosts) have
//     been computed and pushed, then the interior slices, then __syncthreads; barrier.cluster.wait (acquire) only at the
//     start of the next step, so the barrier's latency hides behind the interior work.  Interior slices read no ghost
//     and are no ghost (the spring graph is symmetric), which is what makes the early arrive safe.
//   * Row evaluation and the particle update are the functions of lsm_kernels.cuh (row_forces with GM_SMEM gathers,
//     particle_math): the same arithmetic in the same order as the direct and streamed kernels, so exact mode stays
//     bit-identical to the serial reference.  Breakage marks go to the global lists and to the resident copy.
//   * Only plain time steps run here; sample steps, the last step of an lsm_step call and compaction are the streamed
//     kernel's (one launch each), exactly as for the cooperative multi-step launch.
#pragma once
#include "lsm_kernels.cuh"

namespace lsmk {

constexpr int kResThreads = 512;       // 16 warps, one CTA per SM (the window fills most of its shared memory)
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
__device__ __forceinline__ void st_cluster_d2(uint32_t addr, double2 v) {
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
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
__device__ __forceinline__ uint2 lds_u2(uint32_t addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

template <int PM, bool EXACT>
__global__ void __launch_bounds__(kResThreads, 1) k_resident(const StepParams P, const ResLayout L, const ResParams Q) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    constexpr bool kHasThr = (PM == PM_RCF || PM == PM_KRT_RCF || PM == PM_FULL);
    constexpr bool kHasKR = (PM == PM_FULL);
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ ResCta d;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int nwarps = kResThreads / 32;
    if (tid < (int)(sizeof(ResCta) / 4)) reinterpret_cast<int32_t *>(&d)[tid] = reinterpret_cast<const int32_t *>(Q.desc + blockIdx.x)[tid];
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
        if (kHasThr) res_copy16(smem + L.thr, P.sp.thr + e0, ne * 2, tid);
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
    auto do_slice = [&](int k, uint32_t pc, uint32_t pn, long long step, bool push) {
        const uint2 se = lds_u2(slice_s + (uint32_t)k * 8u);
        const int li = (int)(se.x & 0xFFFFu) * kSlice + lane;     // index among own particles
        if (li >= n_own) return;
        const int p = own_lo + li;
        const unsigned w = se.x >> 16;
        const unsigned rel = se.y * kSlice + lane;
        RowSrc R;
        R.nbr = nullptr;
        R.nbr16 = reinterpret_cast<const int16_t *>(smem + L.nbr) + rel;
        R.thr = reinterpret_cast<const uint16_t *>(smem + L.thr) + rel;
        R.typ = (smem + L.typ) + rel;
        R.kF = reinterpret_cast<const double *>(smem + L.kF) + rel;
        R.r0F = reinterpret_cast<const double *>(smem + L.r0F) + rel;
        R.e0 = (size_t)(slot0 + se.y) * kSlice + lane;
        StepVar V;
        V.pos_cur = nullptr; V.pos_next = nullptr; V.step = step;
        V.pos_s = pc - (uint32_t)wlo * 16u;
        const double2 xp = lds_d2(V.pos_s + (uint32_t)p * 16u);
        const double2 vh = lds_d2(vel_s + (uint32_t)li * 16u);
        const uint8_t g = (uint8_t)lds_u8(grp_s + (uint32_t)li);
        double fx = 0.0, fy = 0.0, uu = 0.0;
        row_forces<PM, EXACT, false, GM_SMEM, true>(P, V, R, s_tab, p, w, xp, fx, fy, uu);
        const Upd o = particle_math<EXACT, true, true, false>(P, step, p, xp, vh, g, fx, fy);
        sts_d2(pn + (uint32_t)(p - wlo) * 16u, o.xn);
        if (g == kFree) sts_d2(vel_s + (uint32_t)li * 16u, o.w);
        if (push) {
            for (int q = 0; q < n_push; ++q)
                if (p >= d.push[q].lo && p < d.push[q].hi)
                    st_cluster_d2(map_to_rank(pn + (uint32_t)(p - d.push[q].rwlo) * 16u, (unsigned)d.push[q].rank), o.xn);
        }
    };

    // ---------------- time steps ----------------
    // Warp w takes entries w, w + 16, ... of the order list: its boundary slices first, then (after arriving on the
    // cluster barrier) its interior ones -- every warp gets the same number of slices (+-1).
    bool cur = false;
    for (int it = 0; it < Q.nsteps; ++it) {
        const bool more = it + 1 < Q.nsteps;
        const uint32_t pc = cur ? posB : posA, pn = cur ? posA : posB;
        if (it > 0) cluster_wait();                            // ghosts of this step have arrived; last step's readers are done
        int k = warp;
        for (; k < n_boundary; k += nwarps) do_slice(k, pc, pn, P.step + it, more);
        __syncwarp();
        if (more) { if (warp < n_boundary) cluster_arrive(); else cluster_arrive_relaxed(); }   // release only what was pushed
        for (; k < n_sl; k += nwarps) do_slice(k, pc, pn, P.step + it, false);
        __syncthreads();                                       // own-region writes of this step before anyone's next step
        cur = !cur;
    }

    // ---------------- store the own particles ----------------
    const double2 *res = reinterpret_cast<const double2 *>(smem + (cur ? L.pos1 : L.pos0)) + (own_lo - wlo);
    for (int i = tid; i < n_own; i += kResThreads) { Q.pos_io[own_lo + i] = res[i]; P.vel[own_lo + i] = s_vel[i]; }
}

}  // namespace lsmk
