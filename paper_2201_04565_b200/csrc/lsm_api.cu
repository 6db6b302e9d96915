// lsm_api.cu -- host side of liblsm_b200.so: the C ABI of include/lsm.h.
// Validation, renumbering (a8), layout construction, the step loop (launch sequencing, fused cooperative launches),
// sampling ring, compaction scheduling, numbering translation at the boundary.  All arithmetic of the method runs in the kernels of
// lsm_kernels.cuh; nothing here computes a force or integrates.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/lsm.h"
#include "lsm_kernels.cuh"
#include "lsm_kernels3.cuh"
#include "lsm_resident.cuh"
#include "lsm_window.cuh"

using namespace lsmk;

static thread_local std::string g_create_error;

namespace {

struct Group {
    bool set = false;
    int mode = 0;
    double du[3] = {0, 0, 0};
    long long n0 = 0;
    std::vector<int32_t> ids;  // internal ids, sorted
    int32_t *d_ids = nullptr;
    long long *d_seg = nullptr;  // [B+1]
};

}  // namespace

struct lsm_sim {
    // configuration
    long long N = 0, M = 0;
    int B = 1, dim = 2;
    double dt = 0, gamma = 0, mass_u = 1;
    int sample_every = 0, hist_cap = 1024, compact_every = 0, reorder = 0, force_mode = LSM_FORCE_GATHER, exact = 0, step_fusion = 0, cluster_size = 0;
    int device = 0;
    cudaStream_t stream = nullptr;
    lsm_alloc_fn alloc = nullptr;
    lsm_free_fn free_ = nullptr;
    void *alloc_user = nullptr;
    std::vector<void *> dev_allocs;
    long long device_bytes = 0;
    // numbering
    std::vector<int32_t> perm, inv;  // internal -> caller, caller -> internal (empty = identity)
    std::vector<long long> poff;
    std::vector<uint8_t> h_grp;      // internal numbering
    int32_t *d_inv = nullptr;
    // device state
    double2 *pos[2] = {nullptr, nullptr}, *vel = nullptr, *f = nullptr, *fd = nullptr, *stage[2] = {nullptr, nullptr};
    double4 *pos3[2] = {nullptr, nullptr}, *vel3 = nullptr, *f3 = nullptr, *fd3 = nullptr;   // dim = 3 (lsm_kernels3.cuh)
    double *stage3[2] = {nullptr, nullptr};                                                  // packed [N*3] staging
    uint8_t *grp = nullptr;
    double *mass = nullptr;
    int cur = 0;
    // gather layout
    long long nslices = 0, E = 0, T = 0, Npad = 0;
    TileHdr *hdr = nullptr;
    int32_t *nbr = nullptr, *sid = nullptr;
    int16_t *nbr16 = nullptr;
    thr_t *thr = nullptr;
    uint32_t thr_base = 0, thr_shift = 0;
    double *rcS = nullptr;
    // repacking stage of the compaction (a7): scan scratch, one scratch array as large as the largest slot array
    uint32_t *rp_new_off = nullptr, *rp_totals = nullptr;
    unsigned long long *rp_state = nullptr;
    unsigned int *rp_ticket = nullptr;
    void *rp_scratch = nullptr;
    long long E0 = 0;                // slots (x 32 entries) allocated at create
    bool E_stale = false;            // the stored-slot count changed on the device since the host last read it
    int gather_variant = 0;          // resolved: 1 direct, 2 streamed
    StageLayout L;
    int stream_smem = 0, stream_grid = 0, stream_ctas_per_sm = 0;
    uint32_t max_tile_slots = 0;
    double *virial = nullptr;        // [N][3] output buffer of lsm_read_virial (allocated on first use)
    // Lagrangian strain (lsm_read_strain): reference positions = the positions given at create, internal numbering, kept on
    // the host and uploaded on first use (callers that never ask pay no device memory), output buffers likewise
    std::vector<double2> h_ref2;
    std::vector<double4> h_ref3;
    double2 *ref2 = nullptr;
    double4 *ref3 = nullptr;
    double *strain = nullptr;
    uint8_t *strain_ok = nullptr;
    int multi_on = 0;                // fuse runs of plain time steps into one cooperative launch
    // windowed streamed kernel (lsm_window.cuh): neighbour ranges of every tile staged in shared memory by the producer
    int win_on = 0, win_cap = 0, win_smem = 0, win_grid = 0;
    StageLayout LW;
    TileWin *d_win = nullptr;
    uint16_t *widx = nullptr;
    int coopwin_on = 0;              // cooperative multi-step launches re-fetch windows instead of gathering from L2 (k_coop_win)
    // cluster-resident stepping (lsm_resident.cuh): one thread-block cluster per unit (specimen / small lattice)
    int res_on = 0, res_cluster = 0, res_grid = 0, res_active_clusters = 0;
    ResLayout RL;
    ResCta *res_desc = nullptr;
    uint16_t *res_order = nullptr;
    long long multi_max = 4096;
    unsigned long long *gbar = nullptr, gbar_base = 0;
    // scatter layout
    long long Ms = 0;
    int32_t *ssi = nullptr, *ssj = nullptr, *ssid = nullptr;
    int scatter_variant = 0;         // 0 one RED per force component (the paper's design), 1 warp-aggregated, 2 shared-memory tiles
    int32_t *s_own_off = nullptr, *s_jl_off = nullptr, *s_jl_idx = nullptr, *s_tile_off = nullptr;
    int scatter_tiles = 0, scatter_tile_smem = 0;
    double *sUs = nullptr;
    long long *d_soff_list = nullptr;
    // parameters
    int pm = PM_UNIFORM, ntypes = 0;
    uint8_t *typ = nullptr;
    double *kF = nullptr, *r0F = nullptr, *rcF = nullptr, *tab = nullptr;
    double k_u = 0, r0_u = 0, rc_u = 0;
    // breakage
    long long *break_step = nullptr;
    unsigned long long *nbroken = nullptr;
    long long *d_poff = nullptr;
    uint8_t *d_broken = nullptr;
    // reductions
    double *sU = nullptr, *sKE = nullptr, *part = nullptr;
    long long nchunks = 0;
    long long *chunk_lo = nullptr, *chunk_hi = nullptr;
    int *spec_chunk_off = nullptr;
    int *flags = nullptr;
    double *cur_U = nullptr, *cur_KE = nullptr;
    // history ring
    long long *hist_step = nullptr, *hist_nb = nullptr;
    double *hist_R = nullptr, *hist_U = nullptr, *hist_KE = nullptr;
    long long hist_head = 0, hist_count = 0;
    // groups
    Group groups[kMaxGroups];
    // run state
    long long step = 0;
    long long kernels_launched = 0;
    long long last_compact_step = 0;
    lsm_status sticky = LSM_OK;
    std::string err;
};

namespace {

lsm_status fail(lsm_sim *s, lsm_status st, const std::string &msg) {
    if (s) { s->sticky = st; s->err = msg; }
    else g_create_error = msg;
    return st;
}

#define CUDA_TRY(s, expr)                                                                          \
    do {                                                                                           \
        cudaError_t _e = (expr);                                                                   \
        if (_e != cudaSuccess)                                                                     \
            return fail((s), LSM_E_CUDA, std::string(#expr) + ": " + cudaGetErrorString(_e));      \
    } while (0)

template <class T> lsm_status dev_alloc(lsm_sim *s, T **out, size_t count) {
    size_t bytes = std::max<size_t>(count, 1) * sizeof(T);
    void *p = nullptr;
    if (s->alloc) {
        p = s->alloc(bytes, s->alloc_user);
        if (!p) return fail(s, LSM_E_NOMEM, "device allocator callback returned NULL");
    } else {
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e != cudaSuccess) return fail(s, e == cudaErrorMemoryAllocation ? LSM_E_NOMEM : LSM_E_CUDA, std::string("cudaMalloc: ") + cudaGetErrorString(e));
    }
    s->dev_allocs.push_back(p);
    s->device_bytes += (long long)bytes;
    *out = reinterpret_cast<T *>(p);
    return LSM_OK;
}

template <class T> lsm_status upload(lsm_sim *s, T **out, const std::vector<T> &h) {
    lsm_status st = dev_alloc(s, out, h.size());
    if (st != LSM_OK) return st;
    if (!h.empty()) CUDA_TRY(s, cudaMemcpyAsync(*out, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, s->stream));
    return LSM_OK;
}

// Return one allocation made through dev_alloc (the caller has made sure no enqueued work still uses it).
void dev_free(lsm_sim *s, void *p) {
    if (!p) return;
    auto it = std::find(s->dev_allocs.begin(), s->dev_allocs.end(), p);
    if (it == s->dev_allocs.end()) return;
    s->dev_allocs.erase(it);
    if (s->alloc) { if (s->free_) s->free_(p, s->alloc_user); }
    else cudaFree(p);
}

// Makes the handle's device current for the duration of an entry point and restores the caller's device afterwards.
struct DeviceScope {
    int prev = -1;
    explicit DeviceScope(int dev) { if (cudaGetDevice(&prev) != cudaSuccess) prev = -1; if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceScope() { if (prev >= 0) cudaSetDevice(prev); }
};

#define TRY(expr)                         \
    do {                                  \
        lsm_status _st = (expr);          \
        if (_st != LSM_OK) return _st;    \
    } while (0)

inline unsigned grid_for(long long n) { return (unsigned)((n + kBlock - 1) / kBlock); }

inline uint64_t part1by1(uint64_t x) {
    x &= 0xffffffffull;
    x = (x | (x << 16)) & 0x0000ffff0000ffffull;
    x = (x | (x << 8)) & 0x00ff00ff00ff00ffull;
    x = (x | (x << 4)) & 0x0f0f0f0f0f0f0f0full;
    x = (x | (x << 2)) & 0x3333333333333333ull;
    x = (x | (x << 1)) & 0x5555555555555555ull;
    return x;
}

// Breakage filter word of a breaking length rc: (high 32 bits of rc*rc) - 1 (lsm_kernels.cuh, row_chunk).
uint32_t thr_of(double rc) {
    const double rc2 = rc * rc;
    uint64_t u; std::memcpy(&u, &rc2, 8);
    const uint32_t hi = (uint32_t)(u >> 32);
    return hi > 0 ? hi - 1 : 0;
}

GroupTab group_tab(const lsm_sim *s) {
    GroupTab g;
    for (int i = 0; i < kMaxGroups; ++i) {
        g.dux[i] = s->groups[i].set ? s->groups[i].du[0] : 0.0;
        g.duy[i] = s->groups[i].set ? s->groups[i].du[1] : 0.0;
        g.duz[i] = s->groups[i].set ? s->groups[i].du[2] : 0.0;
        g.n0[i] = s->groups[i].n0;
    }
    return g;
}

StepParams step_params(const lsm_sim *s, long long step) {
    StepParams P;
    std::memset(&P, 0, sizeof(P));
    const bool gather = s->force_mode == LSM_FORCE_GATHER;
    if (s->dim == 3) {   // the streamed D = 3 instantiation reads these as double4 records (lsm_rows3.cuh)
        P.pos_cur = reinterpret_cast<const double2 *>(s->pos3[s->cur]);
        P.pos_next = reinterpret_cast<double2 *>(s->pos3[s->cur ^ 1]);
        P.vel = reinterpret_cast<double2 *>(s->vel3); P.f = reinterpret_cast<double2 *>(s->f3); P.fd = reinterpret_cast<double2 *>(s->fd3);
    } else {
        P.pos_cur = s->pos[s->cur];
        P.pos_next = gather ? s->pos[s->cur ^ 1] : s->pos[s->cur];
        P.vel = s->vel; P.f = s->f; P.fd = s->fd;
    }
    P.grp = s->grp; P.mass = s->mass;
    P.mass_u = s->mass_u; P.inv_mass_u = 1.0 / s->mass_u;
    P.dt = s->dt; P.hdt = 0.5 * s->dt; P.gamma = s->gamma;
    P.N = s->N; P.step = step;
    P.hdr = s->hdr; P.T = s->T; P.nbr = s->nbr; P.nbr16 = s->nbr16; P.widx = s->widx; P.sid = s->sid;
    P.sp.typ = s->typ; P.sp.kF = s->kF; P.sp.r0F = s->r0F; P.sp.rcF = s->rcF; P.sp.tab = s->tab; P.sp.ntypes = s->ntypes;
    P.sp.thr = s->thr; P.sp.thr_base = s->thr_base; P.sp.thr_mul = 1u << s->thr_shift; P.sp.rcS = s->rcS; P.sp.kr0_u = s->k_u * s->r0_u; P.sp.thr_u = thr_of(s->rc_u);
    P.sp.k_u = s->k_u; P.sp.r0_u = s->r0_u; P.sp.rc_u = s->rc_u;
    P.break_step = s->break_step; P.nbroken = s->nbroken; P.poff = s->d_poff; P.B = s->B;
    P.sU = s->sU; P.sKE = s->sKE;
    P.g = group_tab(s);
    return P;
}

ScatterParams scatter_params(const lsm_sim *s) {
    ScatterParams S;
    std::memset(&S, 0, sizeof(S));
    S.si = s->ssi; S.sj = s->ssj; S.sid = s->ssid; S.M = s->Ms; S.sUs = s->sUs;
    S.own_off = s->s_own_off; S.jl_off = s->s_jl_off; S.jl_idx = s->s_jl_idx; S.tile_off = s->s_tile_off; S.N = s->N;
    S.sp.typ = s->typ; S.sp.kF = s->kF; S.sp.r0F = s->r0F; S.sp.rcF = s->rcF; S.sp.tab = s->tab; S.sp.ntypes = s->ntypes;
    S.sp.k_u = s->k_u; S.sp.r0_u = s->r0_u; S.sp.rc_u = s->rc_u;
    return S;
}

enum Variant { V_MID = 0, V_MID_SAMPLE = 1, V_END = 2, V_INIT = 3 };

GroupTab3 group_tab3(const lsm_sim *s) {
    GroupTab3 g;
    for (int i = 0; i < kMaxGroups; ++i) {
        for (int c = 0; c < 3; ++c) g.du[c][i] = s->groups[i].set ? s->groups[i].du[c] : 0.0;
        g.n0[i] = s->groups[i].n0;
    }
    return g;
}

Step3Params step_params3(const lsm_sim *s, long long step, Variant v) {
    Step3Params P;
    std::memset(&P, 0, sizeof(P));
    const StepParams P2 = step_params(s, step);   // spring layout, parameters and bookkeeping are shared with the 2-D path
    P.pos_cur = s->pos3[s->cur]; P.pos_next = s->pos3[s->cur ^ 1];
    P.vel = s->vel3; P.f = s->f3; P.fd = s->fd3; P.grp = s->grp; P.mass = s->mass; P.mass_u = s->mass_u;
    P.dt = s->dt; P.hdt = 0.5 * s->dt; P.gamma = s->gamma; P.N = s->N; P.step = step;
    P.hdr = s->hdr; P.nbr = s->nbr; P.nbr16 = s->nbr16; P.sid = s->sid; P.sp = P2.sp; P.pm = s->pm;
    P.break_step = s->break_step; P.nbroken = s->nbroken; P.poff = s->d_poff; P.B = s->B; P.sU = s->sU; P.sKE = s->sKE;
    P.kick2 = v != V_INIT; P.advance = v == V_MID || v == V_MID_SAMPLE; P.sample = v != V_MID;
    P.g = group_tab3(s);
    return P;
}

void launch_gather3(lsm_sim *s, long long step, Variant v) {
    const Step3Params P = step_params3(s, step, v);
    if (s->exact) k3_step<true><<<grid_for(s->N), kBlock, 0, s->stream>>>(P);
    else k3_step<false><<<grid_for(s->N), kBlock, 0, s->stream>>>(P);
    s->kernels_launched += 1;
}

template <int PM, bool EXACT> void launch_gather_v(const StepParams &P, Variant v, unsigned grid, cudaStream_t st) {
    switch (v) {
        case V_MID: k_gather_step<PM, EXACT, true, true, false><<<grid, kBlock, 0, st>>>(P); break;
        case V_MID_SAMPLE: k_gather_step<PM, EXACT, true, true, true><<<grid, kBlock, 0, st>>>(P); break;
        case V_END: k_gather_step<PM, EXACT, true, false, true><<<grid, kBlock, 0, st>>>(P); break;
        case V_INIT: k_gather_step<PM, EXACT, false, false, true><<<grid, kBlock, 0, st>>>(P); break;
    }
}

template <bool EXACT> void launch_gather_pm(int pm, const StepParams &P, Variant v, unsigned grid, cudaStream_t st) {
    switch (pm) {
        case PM_UNIFORM: launch_gather_v<PM_UNIFORM, EXACT>(P, v, grid, st); break;
        case PM_TYPED: launch_gather_v<PM_TYPED, EXACT>(P, v, grid, st); break;
        case PM_RCF: launch_gather_v<PM_RCF, EXACT>(P, v, grid, st); break;
        case PM_KRT_RCF: launch_gather_v<PM_KRT_RCF, EXACT>(P, v, grid, st); break;
        default: launch_gather_v<PM_FULL, EXACT>(P, v, grid, st); break;
    }
}

// Opt a kernel in to > 48 KB of dynamic shared memory.  The attribute is per device: remembered per device ordinal.
constexpr int kMaxDevices = 64;
struct OptIn { int bytes[kMaxDevices]; OptIn() { for (int &b : bytes) b = -1; } };
template <class K> void stream_opt_in(K kern, const lsm_sim *s, OptIn &done) {
    int &have = done.bytes[s->device < kMaxDevices ? s->device : kMaxDevices - 1];
    if (have < s->stream_smem || s->device >= kMaxDevices - 1) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, s->stream_smem) == cudaSuccess) have = s->stream_smem;
    }   // a failure shows up as a launch error, which the callers check
}

template <int PM, bool EXACT, bool KICK2, bool ADVANCE, bool SAMPLE> void launch_stream_one(const lsm_sim *s, const StepParams &P) {
    MultiParams M;
    std::memset(&M, 0, sizeof(M));
    if (s->dim == 3) {
        if (s->nbr16) {
            auto kern = k_gather_stream<PM, EXACT, KICK2, ADVANCE, SAMPLE, false, true, 3>;
            static thread_local OptIn configured_for;
            stream_opt_in(kern, s, configured_for);
            kern<<<s->stream_grid, kTile + 32, s->stream_smem, s->stream>>>(P, s->L, M);
        } else {
            auto kern = k_gather_stream<PM, EXACT, KICK2, ADVANCE, SAMPLE, false, false, 3>;
            static thread_local OptIn configured_for;
            stream_opt_in(kern, s, configured_for);
            kern<<<s->stream_grid, kTile + 32, s->stream_smem, s->stream>>>(P, s->L, M);
        }
    } else if (s->nbr16) {
        auto kern = k_gather_stream<PM, EXACT, KICK2, ADVANCE, SAMPLE, false, true>;
        static thread_local OptIn configured_for;
        stream_opt_in(kern, s, configured_for);
        kern<<<s->stream_grid, kTile + 32, s->stream_smem, s->stream>>>(P, s->L, M);
    } else {
        auto kern = k_gather_stream<PM, EXACT, KICK2, ADVANCE, SAMPLE, false, false>;
        static thread_local OptIn configured_for;
        stream_opt_in(kern, s, configured_for);
        kern<<<s->stream_grid, kTile + 32, s->stream_smem, s->stream>>>(P, s->L, M);
    }
}

// nsteps consecutive non-sample time steps in ONE cooperative launch (grid barrier between steps).
template <int PM, bool EXACT> cudaError_t launch_stream_multi_one(const lsm_sim *s, StepParams P, MultiParams M) {
    StageLayout L = s->L;
    void *args[3] = {&P, &L, &M};
    // (a grid the device cannot keep resident makes cudaLaunchCooperativeKernel fail with
    //  cudaErrorCooperativeLaunchTooLarge instead of deadlocking at the grid barrier; lsm_step reports it)
    if (s->dim == 3) {
        if (s->nbr16) {
            auto kern = k_gather_stream<PM, EXACT, true, true, false, true, true, 3>;
            static thread_local OptIn configured_for;
            stream_opt_in(kern, s, configured_for);
            return cudaLaunchCooperativeKernel((const void *)kern, dim3(s->stream_grid), dim3(kTile + 32), args, (size_t)s->stream_smem, s->stream);
        }
        auto kern = k_gather_stream<PM, EXACT, true, true, false, true, false, 3>;
        static thread_local OptIn configured_for;
        stream_opt_in(kern, s, configured_for);
        return cudaLaunchCooperativeKernel((const void *)kern, dim3(s->stream_grid), dim3(kTile + 32), args, (size_t)s->stream_smem, s->stream);
    }
    if (s->nbr16) {
        auto kern = k_gather_stream<PM, EXACT, true, true, false, true, true>;
        static thread_local OptIn configured_for;
        stream_opt_in(kern, s, configured_for);
        return cudaLaunchCooperativeKernel((const void *)kern, dim3(s->stream_grid), dim3(kTile + 32), args, (size_t)s->stream_smem, s->stream);
    }
    auto kern = k_gather_stream<PM, EXACT, true, true, false, true, false>;
    static thread_local OptIn configured_for;
    stream_opt_in(kern, s, configured_for);
    return cudaLaunchCooperativeKernel((const void *)kern, dim3(s->stream_grid), dim3(kTile + 32), args, (size_t)s->stream_smem, s->stream);
}

template <bool EXACT> cudaError_t launch_stream_multi_pm(const lsm_sim *s, const StepParams &P, const MultiParams &M) {
    switch (s->pm) {
        case PM_UNIFORM: return launch_stream_multi_one<PM_UNIFORM, EXACT>(s, P, M);
        case PM_TYPED: return launch_stream_multi_one<PM_TYPED, EXACT>(s, P, M);
        case PM_RCF: return launch_stream_multi_one<PM_RCF, EXACT>(s, P, M);
        case PM_KRT_RCF: return launch_stream_multi_one<PM_KRT_RCF, EXACT>(s, P, M);
        default: return launch_stream_multi_one<PM_FULL, EXACT>(s, P, M);
    }
}

template <int PM, bool EXACT> void launch_stream_v(const lsm_sim *s, const StepParams &P, Variant v) {
    switch (v) {
        case V_MID: launch_stream_one<PM, EXACT, true, true, false>(s, P); break;
        case V_MID_SAMPLE: launch_stream_one<PM, EXACT, true, true, true>(s, P); break;
        case V_END: launch_stream_one<PM, EXACT, true, false, true>(s, P); break;
        case V_INIT: launch_stream_one<PM, EXACT, false, false, true>(s, P); break;
    }
}

template <bool EXACT> void launch_stream_pm(const lsm_sim *s, const StepParams &P, Variant v) {
    switch (s->pm) {
        case PM_UNIFORM: launch_stream_v<PM_UNIFORM, EXACT>(s, P, v); break;
        case PM_TYPED: launch_stream_v<PM_TYPED, EXACT>(s, P, v); break;
        case PM_RCF: launch_stream_v<PM_RCF, EXACT>(s, P, v); break;
        case PM_KRT_RCF: launch_stream_v<PM_KRT_RCF, EXACT>(s, P, v); break;
        default: launch_stream_v<PM_FULL, EXACT>(s, P, v); break;
    }
}

// ---- cluster-resident stepping: plan (host, at create) and launch -------------------------------------------------------
// Splits every unit (specimen) into C contiguous slice ranges, one per CTA of a cluster, and derives each CTA's window
// (own particles + ghosts), the ghost ranges it pushes to the other CTAs, and its boundary-first slice order.
// nbmin / nbmax: smallest / largest neighbour id of every particle (own id where it has none).
struct ResPlan {
    int C = 0;
    std::vector<ResCta> desc;
    std::vector<uint16_t> order;
    ResLayout L;
    bool ok = false;
    int active = 0;              // clusters of this shape the device holds at once (cudaOccupancyMaxActiveClusters)
};

ResPlan plan_resident(const lsm_sim *s, int C, const std::vector<int32_t> &nbmin, const std::vector<int32_t> &nbmax,
                      const std::vector<uint32_t> &off, int smem_budget) {
    ResPlan R;
    R.C = C;
    std::memset(&R.L, 0, sizeof(R.L));
    const int B = s->B;
    R.desc.assign((size_t)B * C, ResCta{});
    std::vector<std::vector<uint16_t>> ord((size_t)B * C);
    long long win_cap = 0, sl_cap = 0, slot_cap = 0;
    for (int b = 0; b < B; ++b) {
        const long long u0 = s->poff[b], u1 = s->poff[b + 1];
        if (u0 % kSlice) return R;                                    // units must start on a slice boundary
        const long long S0 = u0 / kSlice, S1 = (u1 + kSlice - 1) / kSlice, nsu = S1 - S0;
        const long long base = nsu / C, rem = nsu % C;
        ResCta *dd = &R.desc[(size_t)b * C];
        for (int c = 0; c < C; ++c) {
            const long long a = S0 + c * base + std::min<long long>(c, rem), e = a + base + (c < rem ? 1 : 0);
            ResCta &q = dd[c];
            q.sl0 = (int32_t)a; q.n_sl = (int32_t)(e - a);
            q.own_lo = (int32_t)(a * kSlice);
            q.n_own = (int32_t)std::max<long long>(0, std::min<long long>(u1, e * kSlice) - a * kSlice);
            long long lo = q.own_lo, hi = (long long)q.own_lo + q.n_own;
            for (long long p = q.own_lo; p < (long long)q.own_lo + q.n_own; ++p) { lo = std::min<long long>(lo, nbmin[p]); hi = std::max<long long>(hi, (long long)nbmax[p] + 1); }
            q.wlo = (int32_t)lo; q.wlen = (int32_t)(hi - lo);
            win_cap = std::max<long long>(win_cap, q.wlen);
            sl_cap = std::max<long long>(sl_cap, q.n_sl);
            slot_cap = std::max<long long>(slot_cap, (long long)off[e] - (long long)off[a]);
        }
        for (int c = 0; c < C; ++c) {   // ghost ranges: my own particles inside another CTA's window
            ResCta &q = dd[c];
            q.n_push = 0;
            const long long o0 = q.own_lo, o1 = (long long)q.own_lo + q.n_own;
            for (int r = 0; r < C; ++r) {
                if (r == c || dd[r].wlen == 0) continue;
                const long long lo = std::max<long long>(o0, dd[r].wlo), hi = std::min<long long>(o1, (long long)dd[r].wlo + dd[r].wlen);
                if (lo >= hi) continue;
                if (q.n_push == kResMaxPush) return R;               // numbering not banded enough for this cluster size
                q.push[q.n_push++] = ResPush{r, (int32_t)lo, (int32_t)hi, dd[r].wlo};
            }
            std::vector<uint16_t> bnd, inner;   // boundary slices (exchange ghosts either way) first
            for (int ls = 0; ls < q.n_sl; ++ls) {
                const long long p0 = o0 + (long long)ls * kSlice, p1 = std::min<long long>(o1, p0 + kSlice);
                bool bd = false;
                for (int k = 0; k < q.n_push && !bd; ++k) bd = p0 < q.push[k].hi && q.push[k].lo < p1;
                for (long long p = p0; p < p1 && !bd; ++p) bd = nbmin[p] < o0 || nbmax[p] >= o1;
                (bd ? bnd : inner).push_back((uint16_t)ls);
            }
            q.n_boundary = (int32_t)bnd.size();
            bnd.insert(bnd.end(), inner.begin(), inner.end());
            ord[(size_t)b * C + c].swap(bnd);
        }
        // The ghost exchange is safe only when pushes are mutual: a CTA waits, per step, for the pushes of exactly the CTAs
        // it pushes to, and that wait is what keeps a neighbour from running two steps ahead and landing step n+2 ghosts on
        // a transaction barrier whose step-n phase is still open.  Windows are id hulls, so on an irregular graph (a band
        // plus a few long springs) CTA r can lie inside hull(c) without any spring into c: c pushes to r, r not to c.
        // Lattices and banded numberings always give mutual pushes; anything else is not planned as resident.
        for (int c = 0; c < C; ++c)
            for (int k = 0; k < dd[c].n_push; ++k) {
                const ResCta &t = dd[dd[c].push[k].rank];
                bool back = false;
                for (int m = 0; m < t.n_push && !back; ++m) back = t.push[m].rank == c;
                if (!back) return R;
            }
    }
    if (sl_cap > 65535) return R;
    const bool need_typ = s->pm == PM_TYPED || s->pm == PM_KRT_RCF, need_thr = s->pm == PM_RCF || s->pm == PM_KRT_RCF || s->pm == PM_FULL, need_kr = s->pm == PM_FULL;
    ResLayout &L = R.L;
    auto up = [](long long x) { return (x + 127) & ~127LL; };
    long long o = 0;
    L.tab = (int)o; if (need_typ) o += up((long long)s->ntypes * kTabStride * 8);
    L.win_cap = (int)win_cap; L.sl_cap = (int)std::max<long long>(sl_cap, 1); L.own_cap = (int)(sl_cap * kSlice); L.slot_cap = (int)slot_cap;
    L.pos0 = (int)o; o += up(win_cap * 16);
    L.pos1 = (int)o; o += up(win_cap * 16);
    L.vel = (int)o; o += up(sl_cap * kSlice * 16);
    L.grp = (int)o; o += up(sl_cap * kSlice);
    L.sl_off = (int)o; o += up(sl_cap * 8);        // {slice | width << 16, slot offset} per entry of the order list
    L.nbr = (int)o; o += up(slot_cap * kSlice * 2);
    L.thr = (int)o; if (need_thr) o += up(slot_cap * kSlice * kThrB);
    L.typ = (int)o; if (need_typ) o += up(slot_cap * kSlice);
    L.kF = (int)o; if (need_kr) o += up(slot_cap * kSlice * 8);
    L.r0F = (int)o; if (need_kr) o += up(slot_cap * kSlice * 8);
    if (o > smem_budget) return R;
    L.bytes = (int)o;
    R.order.assign((size_t)B * C * L.sl_cap, 0);
    for (size_t i = 0; i < ord.size(); ++i) std::copy(ord[i].begin(), ord[i].end(), R.order.begin() + i * L.sl_cap);
    R.ok = true;
    return R;
}

// Opt the resident kernel in to `bytes` of dynamic shared memory and to non-portable cluster sizes, once per device and
// size.  The attribute is only ever raised: the occupancy queries at create ask about several candidate layouts in turn.
template <int PM, bool EXACT> cudaError_t resident_configure(const lsm_sim *s, int bytes) {
    auto kern = k_resident<PM, EXACT>;
    static thread_local OptIn configured_for;
    int &have = configured_for.bytes[s->device < kMaxDevices ? s->device : kMaxDevices - 1];
    if (have < bytes || s->device >= kMaxDevices - 1) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
        have = bytes;
    }
    return cudaSuccess;
}

template <int PM, bool EXACT> cudaError_t launch_resident_one(const lsm_sim *s, const StepParams &P, const ResParams &Q) {
    auto kern = k_resident<PM, EXACT>;
    cudaError_t e0 = resident_configure<PM, EXACT>(s, s->RL.bytes);
    if (e0 != cudaSuccess) return e0;
    cudaLaunchConfig_t cfg;
    std::memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)s->res_grid); cfg.blockDim = dim3(kResThreads); cfg.dynamicSmemBytes = (size_t)s->RL.bytes; cfg.stream = s->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)s->res_cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, P, s->RL, Q);
}

// How many clusters of C CTAs with `bytes` of dynamic shared memory each the current device can hold at once (0: such a
// cluster cannot be scheduled here at all -- a MIG slice, a GPC with too few free SMs, a smaller part).  Asked at create.
template <int PM, bool EXACT> int resident_clusters_one(const lsm_sim *s, int C, int bytes) {
    auto kern = k_resident<PM, EXACT>;
    if (resident_configure<PM, EXACT>(s, bytes) != cudaSuccess) { cudaGetLastError(); return 0; }
    cudaLaunchConfig_t cfg;
    std::memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)C); cfg.blockDim = dim3(kResThreads); cfg.dynamicSmemBytes = (size_t)bytes;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
    return n;
}

int resident_clusters(const lsm_sim *s, int C, int bytes) {
    switch (s->pm) {
        case PM_UNIFORM: return s->exact ? resident_clusters_one<PM_UNIFORM, true>(s, C, bytes) : resident_clusters_one<PM_UNIFORM, false>(s, C, bytes);
        case PM_TYPED: return s->exact ? resident_clusters_one<PM_TYPED, true>(s, C, bytes) : resident_clusters_one<PM_TYPED, false>(s, C, bytes);
        case PM_RCF: return s->exact ? resident_clusters_one<PM_RCF, true>(s, C, bytes) : resident_clusters_one<PM_RCF, false>(s, C, bytes);
        case PM_KRT_RCF: return s->exact ? resident_clusters_one<PM_KRT_RCF, true>(s, C, bytes) : resident_clusters_one<PM_KRT_RCF, false>(s, C, bytes);
        default: return s->exact ? resident_clusters_one<PM_FULL, true>(s, C, bytes) : resident_clusters_one<PM_FULL, false>(s, C, bytes);
    }
}

template <bool EXACT> cudaError_t launch_resident_pm(const lsm_sim *s, const StepParams &P, const ResParams &Q) {
    switch (s->pm) {
        case PM_UNIFORM: return launch_resident_one<PM_UNIFORM, EXACT>(s, P, Q);
        case PM_TYPED: return launch_resident_one<PM_TYPED, EXACT>(s, P, Q);
        case PM_RCF: return launch_resident_one<PM_RCF, EXACT>(s, P, Q);
        case PM_KRT_RCF: return launch_resident_one<PM_KRT_RCF, EXACT>(s, P, Q);
        default: return launch_resident_one<PM_FULL, EXACT>(s, P, Q);
    }
}

template <int PM, bool EXACT> void launch_win_one(const lsm_sim *s, const StepParams &P, const WinParams &W) {
    auto kern = k_gather_win<PM, EXACT>;
    static thread_local OptIn configured_for;
    int &have = configured_for.bytes[s->device < kMaxDevices ? s->device : kMaxDevices - 1];
    if (have < s->win_smem || s->device >= kMaxDevices - 1) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, s->win_smem) == cudaSuccess) have = s->win_smem;
    }
    kern<<<s->win_grid, kTile + 32, s->win_smem, s->stream>>>(P, s->LW, W);
}

template <bool EXACT> void launch_win_pm(const lsm_sim *s, const StepParams &P, const WinParams &W) {
    switch (s->pm) {
        case PM_UNIFORM: launch_win_one<PM_UNIFORM, EXACT>(s, P, W); break;
        case PM_TYPED: launch_win_one<PM_TYPED, EXACT>(s, P, W); break;
        case PM_RCF: launch_win_one<PM_RCF, EXACT>(s, P, W); break;
        case PM_KRT_RCF: launch_win_one<PM_KRT_RCF, EXACT>(s, P, W); break;
        default: launch_win_one<PM_FULL, EXACT>(s, P, W); break;
    }
}

template <int PM, bool EXACT> cudaError_t launch_coopwin_one(const lsm_sim *s, StepParams P, CoopWinParams Q) {
    auto kern = k_coop_win<PM, EXACT>;
    static thread_local OptIn configured_for;
    int &have = configured_for.bytes[s->device < kMaxDevices ? s->device : kMaxDevices - 1];
    if (have < s->win_smem || s->device >= kMaxDevices - 1) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, s->win_smem) == cudaSuccess) have = s->win_smem;
    }
    StageLayout L = s->LW;
    void *args[3] = {&P, &L, &Q};
    return cudaLaunchCooperativeKernel((const void *)kern, dim3(s->win_grid), dim3(kTile + 32), args, (size_t)s->win_smem, s->stream);
}

template <bool EXACT> cudaError_t launch_coopwin_pm(const lsm_sim *s, const StepParams &P, const CoopWinParams &Q) {
    switch (s->pm) {
        case PM_UNIFORM: return launch_coopwin_one<PM_UNIFORM, EXACT>(s, P, Q);
        case PM_TYPED: return launch_coopwin_one<PM_TYPED, EXACT>(s, P, Q);
        case PM_RCF: return launch_coopwin_one<PM_RCF, EXACT>(s, P, Q);
        case PM_KRT_RCF: return launch_coopwin_one<PM_KRT_RCF, EXACT>(s, P, Q);
        default: return launch_coopwin_one<PM_FULL, EXACT>(s, P, Q);
    }
}

// nsteps plain time steps, first force evaluation = step `step`, state resident in the clusters' shared memory.
cudaError_t launch_resident(lsm_sim *s, long long step, int nsteps) {
    const StepParams P = step_params(s, step);
    ResParams Q;
    Q.desc = s->res_desc; Q.order = s->res_order; Q.pos_io = s->pos[s->cur]; Q.nsteps = nsteps;
    return s->exact ? launch_resident_pm<true>(s, P, Q) : launch_resident_pm<false>(s, P, Q);
}

void launch_gather(lsm_sim *s, const StepParams &P, Variant v) {
    if (s->dim == 3 && s->gather_variant != 2) { launch_gather3(s, P.step, v); return; }
    if (s->win_on && v == V_MID) {       // plain time step: neighbour windows staged by the producer, gathers from shared memory
        WinParams W;
        W.win = s->d_win; W.widx = s->widx; W.win_off = s->LW.pos;
        if (s->exact) launch_win_pm<true>(s, P, W); else launch_win_pm<false>(s, P, W);
    } else if (s->gather_variant == 2) {
        if (s->exact) launch_stream_pm<true>(s, P, v);
        else launch_stream_pm<false>(s, P, v);
    } else {
        const unsigned grid = (unsigned)s->T;
        if (s->exact) launch_gather_pm<true>(s->pm, P, v, grid, s->stream);
        else launch_gather_pm<false>(s->pm, P, v, grid, s->stream);
    }
    s->kernels_launched += 1;
}

template <int PM, bool SAMPLE> void launch_scatter_one(const lsm_sim *s, const StepParams &P, const ScatterParams &S) {
    if (S.M == 0) return;
    if (s->scatter_variant == 1) k_spring_scatter_warp<PM, SAMPLE><<<grid_for(S.M), kBlock, 0, s->stream>>>(P, S);
    else if (s->scatter_variant == 2) {
        auto kern = k_spring_scatter_tile<PM, SAMPLE>;
        static thread_local OptIn configured_for;    // opt in once per device and size, as the other kernels do (static + dynamic may pass 48 KB)
        int &have = configured_for.bytes[s->device < kMaxDevices ? s->device : kMaxDevices - 1];
        if (s->scatter_tile_smem > 32 * 1024 && (have < s->scatter_tile_smem || s->device >= kMaxDevices - 1)) {
            if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, s->scatter_tile_smem) == cudaSuccess) have = s->scatter_tile_smem;
        }   // a failure shows up as a launch error, which the callers check
        kern<<<(unsigned)s->scatter_tiles, kScatterTileThreads, (size_t)s->scatter_tile_smem, s->stream>>>(P, S);
    }
    else k_spring_scatter<PM, SAMPLE><<<grid_for(S.M), kBlock, 0, s->stream>>>(P, S);
}

template <int PM> void launch_scatter_pm(const lsm_sim *s, const StepParams &P, const ScatterParams &S, bool sample) {
    if (sample) launch_scatter_one<PM, true>(s, P, S); else launch_scatter_one<PM, false>(s, P, S);
}

void launch_scatter_force(lsm_sim *s, const StepParams &P, bool sample) {
    const ScatterParams S = scatter_params(s);
    switch (s->pm) {
        case PM_UNIFORM: launch_scatter_pm<PM_UNIFORM>(s, P, S, sample); break;
        case PM_TYPED: launch_scatter_pm<PM_TYPED>(s, P, S, sample); break;
        case PM_RCF: launch_scatter_pm<PM_RCF>(s, P, S, sample); break;
        case PM_KRT_RCF: launch_scatter_pm<PM_KRT_RCF>(s, P, S, sample); break;
        default: launch_scatter_pm<PM_FULL>(s, P, S, sample); break;
    }
    s->kernels_launched += 1;
}

void launch_integrate(lsm_sim *s, const StepParams &P, Variant v) {
    const unsigned grid = grid_for(s->N);
    switch (v) {
        case V_MID: k_integrate<true, true, false><<<grid, kBlock, 0, s->stream>>>(P); break;
        case V_MID_SAMPLE: k_integrate<true, true, true><<<grid, kBlock, 0, s->stream>>>(P); break;
        case V_END: k_integrate<true, false, true><<<grid, kBlock, 0, s->stream>>>(P); break;
        case V_INIT: k_integrate<false, false, true><<<grid, kBlock, 0, s->stream>>>(P); break;
    }
    s->kernels_launched += 1;
}

ReduceParams reduce_params(const lsm_sim *s, long long step) {
    ReduceParams R;
    std::memset(&R, 0, sizeof(R));
    R.sU = s->sU; R.sKE = s->sKE; R.f = s->f;
    R.chunk_lo = s->chunk_lo; R.chunk_hi = s->chunk_hi; R.spec_chunk_off = s->spec_chunk_off; R.part = s->part;
    for (int g = 0; g < kMaxGroups; ++g) {
        R.gids[g] = s->groups[g].set ? s->groups[g].d_ids : nullptr;
        R.gseg[g] = s->groups[g].set ? s->groups[g].d_seg : nullptr;
    }
    R.nbroken = s->nbroken; R.B = s->B; R.step = step; R.flags = s->flags;
    if (s->force_mode == LSM_FORCE_SCATTER) { R.sUs = s->sUs; R.soff_list = s->d_soff_list; }
    return R;
}

// Run the two reduction kernels; slot >= 0 records into the history ring, slot < 0 into cur_U / cur_KE.
void launch_reduce(lsm_sim *s, long long step, long long slot) {
    ReduceParams R = reduce_params(s, step);
    if (slot >= 0) {
        R.out_step = s->hist_step + slot;
        R.out_R = s->hist_R + (size_t)slot * s->B * kMaxGroups * s->dim;
        R.out_U = s->hist_U + (size_t)slot * s->B;
        R.out_KE = s->hist_KE + (size_t)slot * s->B;
        R.out_nb = s->hist_nb + (size_t)slot * s->B;
    } else {
        R.out_U = s->cur_U; R.out_KE = s->cur_KE;
    }
    k_reduce_chunks<<<(unsigned)s->nchunks, kBlock, 0, s->stream>>>(R);
    if (s->dim == 3) {
        Reduce3Params Q;
        Q.R = R; Q.f3 = s->f3; Q.out_R3 = R.out_R; Q.R.out_R = nullptr;
        k3_finalize_sample<<<(unsigned)s->B, kBlock, 0, s->stream>>>(Q);
    } else {
        k_finalize_sample<<<(unsigned)s->B, kBlock, 0, s->stream>>>(R);
    }
    s->kernels_launched += 2;
}

void record_sample(lsm_sim *s, long long step) {
    const long long slot = s->hist_head;
    launch_reduce(s, step, slot);
    s->hist_head = (s->hist_head + 1) % s->hist_cap;
    if (s->hist_count < s->hist_cap) s->hist_count += 1;
}

bool is_sample_step(const lsm_sim *s, long long step) { return s->sample_every > 0 && step > 0 && step % s->sample_every == 0; }

// Force evaluation at the current positions for the current step, without a kick (create / write_state).
lsm_status eval_initial(lsm_sim *s) {
    StepParams P = step_params(s, s->step);
    if (s->force_mode == LSM_FORCE_GATHER) {
        launch_gather(s, P, V_INIT);
    } else {
        k_zero_f<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->f, s->N);
        s->kernels_launched += 1;
        launch_scatter_force(s, P, true);
        launch_integrate(s, P, V_INIT);
    }
    CUDA_TRY(s, cudaGetLastError());
    return LSM_OK;
}

template <class T> void repack_array(lsm_sim *s, const RepackParams &R, T *arr) {
    if (!arr) return;
    T *tmp = reinterpret_cast<T *>(s->rp_scratch);
    k_repack_move<T><<<grid_for(R.nsl * kSlice), kBlock, 0, s->stream>>>(R, arr, tmp);
    k_copy_back<T><<<2048, kBlock, 0, s->stream>>>(R, tmp, arr);
    s->kernels_launched += 2;
}

lsm_status do_compact(lsm_sim *s) {
    if (s->force_mode == LSM_FORCE_GATHER && s->E0 > 0) {
        CompactParams C;
        C.hdr = s->hdr; C.nbr = s->nbr; C.nbr16 = s->nbr16; C.sid = s->sid; C.typ = s->typ; C.thr = s->thr;
        C.kF = s->kF; C.r0F = s->r0F; C.nslices = s->nslices; C.widx = s->widx;
        k_compact_ell<<<grid_for(s->nslices * kSlice), kBlock, 0, s->stream>>>(C);
        s->kernels_launched += 1;
        CUDA_TRY(s, cudaGetLastError());
        // repack: new slot offsets by a device-side scan of the live widths, stable move of every slot array
        const long long nsl = s->T * kTileSlices;
        const long long nblk = (nsl + kBlock - 1) / kBlock;
        if (!s->rp_new_off) {
            TRY(dev_alloc(s, &s->rp_new_off, (size_t)nsl + 1));
            TRY(dev_alloc(s, &s->rp_state, (size_t)nblk));
            TRY(dev_alloc(s, &s->rp_ticket, 1));
            unsigned char *scr = nullptr;
            TRY(dev_alloc(s, &scr, (size_t)s->E0 * kSlice * (s->kF ? 8 : 4)));
            s->rp_scratch = scr;
        }
        RepackParams R;
        R.hdr = s->hdr; R.nsl = nsl; R.new_off = s->rp_new_off; R.state = s->rp_state; R.ticket = s->rp_ticket; R.totals = s->rp_totals;
        CUDA_TRY(s, cudaMemsetAsync(s->rp_state, 0, sizeof(unsigned long long) * nblk, s->stream));
        CUDA_TRY(s, cudaMemsetAsync(s->rp_ticket, 0, sizeof(unsigned int), s->stream));
        k_scan_widths<<<(unsigned)nblk, kBlock, 0, s->stream>>>(R);
        s->kernels_launched += 1;
        repack_array(s, R, s->nbr); repack_array(s, R, s->sid); repack_array(s, R, s->nbr16); repack_array(s, R, s->widx);
        repack_array(s, R, s->typ); repack_array(s, R, s->thr); repack_array(s, R, s->kF); repack_array(s, R, s->r0F);
        k_commit_offsets<<<grid_for(s->T), kBlock, 0, s->stream>>>(R);
        k_commit_total<<<1, 1, 0, s->stream>>>(s->rp_totals);
        s->kernels_launched += 2;
        s->E_stale = true;
        CUDA_TRY(s, cudaGetLastError());
    }
    s->last_compact_step = s->step;
    return LSM_OK;
}

}  // namespace

// =====================================================================================================================
extern "C" {

int32_t lsm_abi_version(void) { return LSM_ABI_VERSION; }

const char *lsm_last_error(const lsm_sim *sim) { return sim ? sim->err.c_str() : g_create_error.c_str(); }

void lsm_destroy(lsm_sim *s) {
    if (!s) return;
    cudaSetDevice(s->device);
    cudaStreamSynchronize(s->stream);
    for (void *p : s->dev_allocs) {
        if (s->alloc) { if (s->free_) s->free_(p, s->alloc_user); }
        else cudaFree(p);
    }
    delete s;
}

static lsm_status create_impl(const lsm_desc *d, lsm_sim *s) {
    const long long N = d->n_particles, M = d->n_springs;
    const int B = d->n_batch;
    s->N = N; s->M = M; s->B = B; s->dim = d->dim; s->dt = d->dt; s->gamma = d->gamma;
    const int D = d->dim;
    s->mass_u = d->mass ? 1.0 : d->mass_uniform;
    s->sample_every = d->sample_every; s->hist_cap = d->history_capacity > 0 ? d->history_capacity : 1024;
    s->compact_every = d->compact_every; s->reorder = d->reorder;
    s->force_mode = d->force_mode == LSM_FORCE_AUTO ? LSM_FORCE_GATHER : d->force_mode;
    if (d->force_mode == LSM_FORCE_SCATTER_WARP) { s->force_mode = LSM_FORCE_SCATTER; s->scatter_variant = 1; }
    if (d->force_mode == LSM_FORCE_SCATTER_TILE) { s->force_mode = LSM_FORCE_SCATTER; s->scatter_variant = 2; }
    s->exact = d->exact; s->step_fusion = d->step_fusion; s->cluster_size = d->cluster_size; s->gather_variant = d->gather_variant; s->device = d->device; s->stream = (cudaStream_t)d->stream;
    s->alloc = d->alloc; s->free_ = d->free_; s->alloc_user = d->alloc_user;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) return fail(s, LSM_E_CUDA, "no CUDA device: this library has no CPU fallback");
    if (d->device < 0 || d->device >= ndev) return fail(s, LSM_E_INVALID, "device ordinal out of range");
    CUDA_TRY(s, cudaSetDevice(d->device));

    // ---- specimen offsets ----
    s->poff.assign(B + 1, 0);
    std::vector<long long> soff(B + 1, 0);
    if (d->particle_offsets && d->spring_offsets) {
        for (int b = 0; b <= B; ++b) { s->poff[b] = d->particle_offsets[b]; soff[b] = d->spring_offsets[b]; }
    } else if (B == 1) { s->poff[1] = N; soff[1] = M; }
    else return fail(s, LSM_E_INVALID, "n_batch > 1 needs particle_offsets and spring_offsets");
    if (s->poff[0] != 0 || s->poff[B] != N || soff[0] != 0 || soff[B] != M) return fail(s, LSM_E_INVALID, "offsets must start at 0 and end at N / M");
    for (int b = 0; b < B; ++b)
        if (s->poff[b + 1] < s->poff[b] || soff[b + 1] < soff[b]) return fail(s, LSM_E_INVALID, "offsets must ascend");

    // ---- validation of values ----
    for (long long q = 0; q < D * N; ++q) {
        if (!std::isfinite(d->x[q])) return fail(s, LSM_E_NONFINITE, "non-finite position");
        if (d->v && !std::isfinite(d->v[q])) return fail(s, LSM_E_NONFINITE, "non-finite velocity");
    }
    if (d->mass) { for (long long p = 0; p < N; ++p) if (!(d->mass[p] > 0.0) || !std::isfinite(d->mass[p])) return fail(s, LSM_E_NONFINITE, "mass must be finite and > 0"); }
    else if (!(d->mass_uniform > 0.0) || !std::isfinite(d->mass_uniform)) return fail(s, LSM_E_NONFINITE, "mass_uniform must be finite and > 0");
    if (M > 0 && (!d->spring_i || !d->spring_j)) return fail(s, LSM_E_INVALID, "spring_i / spring_j are NULL");
    {
        int b = 0;
        for (long long e = 0; e < M; ++e) {
            while (e >= soff[b + 1]) ++b;
            const long long i = d->spring_i[e], j = d->spring_j[e];
            if (i < s->poff[b] || i >= s->poff[b + 1] || j < s->poff[b] || j >= s->poff[b + 1] || i == j)
                return fail(s, LSM_E_RANGE, "spring " + std::to_string(e) + ": endpoint out of its specimen's range, or i == j");
            const double k = d->k ? d->k[e] : d->k_uniform, r0 = d->r0 ? d->r0[e] : d->r0_uniform, rc = d->rc ? d->rc[e] : d->rc_uniform;
            if (!std::isfinite(k) || !std::isfinite(r0) || !std::isfinite(rc) || k < 0.0 || !(r0 > 0.0) || !(rc > 0.0))
                return fail(s, LSM_E_NONFINITE, "spring " + std::to_string(e) + ": need finite k >= 0, r0 > 0, rc > 0");
        }
    }

    // ---- (a8) renumbering: Morton order of the initial positions, per specimen ----
    if (s->reorder == LSM_REORDER_MORTON) {
        s->perm.resize(N); s->inv.resize(N);
        std::vector<std::pair<uint64_t, int32_t>> keys(N);
        for (int b = 0; b < B; ++b) {
            double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
            for (long long p = s->poff[b]; p < s->poff[b + 1]; ++p)
                for (int c = 0; c < D; ++c) { lo[c] = std::min(lo[c], d->x[D * p + c]); hi[c] = std::max(hi[c], d->x[D * p + c]); }
            double ext = 1e-300;
            for (int c = 0; c < D; ++c) ext = std::max(ext, hi[c] - lo[c]);
            const double sc = 1048575.0 / ext;  // 20 bits per axis
            for (long long p = s->poff[b]; p < s->poff[b + 1]; ++p) {
                uint64_t key = 0;
                if (D == 2) {
                    key = part1by1((uint64_t)((d->x[2 * p] - lo[0]) * sc)) | (part1by1((uint64_t)((d->x[2 * p + 1] - lo[1]) * sc)) << 1);
                } else {   // 3-way bit interleave
                    uint64_t q[3];
                    for (int c = 0; c < 3; ++c) q[c] = (uint64_t)((d->x[3 * p + c] - lo[c]) * sc);
                    for (int bit = 0; bit < 20; ++bit)
                        for (int c = 0; c < 3; ++c) key |= ((q[c] >> bit) & 1ull) << (3 * bit + c);
                }
                keys[p] = {key, (int32_t)p};
            }
            std::sort(keys.begin() + s->poff[b], keys.begin() + s->poff[b + 1]);
        }
        for (long long p = 0; p < N; ++p) { s->perm[p] = keys[p].second; s->inv[keys[p].second] = (int32_t)p; }
    }
    // ---- (a8) renumbering: blocked -- bins of ~32 x 8 particles (x by y), bins in row-major order, row-major inside ----
    if (s->reorder == LSM_REORDER_BLOCKED) {
        s->perm.resize(N); s->inv.resize(N);
        struct Key { uint32_t bin; float y, x; int32_t id; };
        std::vector<Key> keys(N);
        for (int b = 0; b < B; ++b) {
            const long long lo_p = s->poff[b], hi_p = s->poff[b + 1];
            if (hi_p == lo_p) continue;
            double lo[2] = {1e300, 1e300}, hi[2] = {-1e300, -1e300};
            for (long long p = lo_p; p < hi_p; ++p)
                for (int c = 0; c < 2; ++c) { lo[c] = std::min(lo[c], d->x[2 * p + c]); hi[c] = std::max(hi[c], d->x[2 * p + c]); }
            const double area = std::max((hi[0] - lo[0]) * (hi[1] - lo[1]), 1e-300);
            const double sp = std::sqrt(area / (double)(hi_p - lo_p));           // mean spacing
            const double wx = 32.0 * sp, wy = 8.0 * sp;
            const uint32_t nbx = (uint32_t)std::min(65535.0, std::floor((hi[0] - lo[0]) / wx) + 1.0);
            for (long long p = lo_p; p < hi_p; ++p) {
                const uint32_t bx = (uint32_t)std::min(65535.0, (d->x[2 * p] - lo[0]) / wx), by = (uint32_t)std::min(65535.0, (d->x[2 * p + 1] - lo[1]) / wy);
                keys[p] = {by * nbx + bx, (float)d->x[2 * p + 1], (float)d->x[2 * p], (int32_t)p};
            }
            std::sort(keys.begin() + lo_p, keys.begin() + hi_p, [](const Key &a, const Key &c) {
                if (a.bin != c.bin) return a.bin < c.bin;
                if (a.y != c.y) return a.y < c.y;
                if (a.x != c.x) return a.x < c.x;
                return a.id < c.id;
            });
        }
        for (long long p = 0; p < N; ++p) { s->perm[p] = keys[p].id; s->inv[keys[p].id] = (int32_t)p; }
    }
    // ---- (a8) renumbering: reverse Cuthill-McKee on the spring graph, per specimen (no coordinates needed) ----
    if (s->reorder == LSM_REORDER_RCM) {
        std::vector<int64_t> aoff(N + 1, 0);
        for (long long e = 0; e < M; ++e) { aoff[d->spring_i[e] + 1]++; aoff[d->spring_j[e] + 1]++; }
        for (long long p = 0; p < N; ++p) aoff[p + 1] += aoff[p];
        std::vector<int32_t> adj(2 * M);
        {
            std::vector<int64_t> fill(aoff.begin(), aoff.end() - 1);
            for (long long e = 0; e < M; ++e) { adj[fill[d->spring_i[e]]++] = d->spring_j[e]; adj[fill[d->spring_j[e]]++] = d->spring_i[e]; }
        }
        auto degree = [&](int32_t p) { return (int64_t)(aoff[p + 1] - aoff[p]); };
        s->perm.assign(N, 0); s->inv.assign(N, 0);
        std::vector<uint8_t> seen(N, 0);
        std::vector<int32_t> order; order.reserve(N);
        std::vector<int32_t> nbrs;
        for (int b = 0; b < B; ++b) {
            const long long lo = s->poff[b], hi = s->poff[b + 1];
            const size_t first = order.size();
            // components in ascending order of their minimum-degree unvisited start (ties: lowest id)
            std::vector<int32_t> starts(hi - lo);
            for (long long p = lo; p < hi; ++p) starts[p - lo] = (int32_t)p;
            std::stable_sort(starts.begin(), starts.end(), [&](int32_t x, int32_t y) { return degree(x) < degree(y); });
            for (int32_t st : starts) {
                if (seen[st]) continue;
                size_t head = order.size();
                order.push_back(st); seen[st] = 1;
                while (head < order.size()) {   // breadth-first, neighbours by ascending degree
                    const int32_t p = order[head++];
                    nbrs.clear();
                    for (int64_t q = aoff[p]; q < aoff[p + 1]; ++q) if (!seen[adj[q]]) { seen[adj[q]] = 1; nbrs.push_back(adj[q]); }
                    std::sort(nbrs.begin(), nbrs.end(), [&](int32_t x, int32_t y) { return degree(x) != degree(y) ? degree(x) < degree(y) : x < y; });
                    order.insert(order.end(), nbrs.begin(), nbrs.end());
                }
            }
            std::reverse(order.begin() + first, order.end());   // the "reverse" of RCM, inside the specimen's id range
        }
        for (long long p = 0; p < N; ++p) { s->perm[p] = order[p]; s->inv[order[p]] = (int32_t)p; }
    }
    auto to_int = [&](long long c) -> int32_t { return s->inv.empty() ? (int32_t)c : s->inv[c]; };

    // ---- parameter encoding: uniform scalars, a type table (Table 1) or fp64 arrays ----
    const bool k_arr = d->k != nullptr, r0_arr = d->r0 != nullptr, rc_arr = d->rc != nullptr;
    std::vector<uint8_t> stype;  // per spring type index
    std::vector<double> tab;
    {
        auto all_same = [&](const double *a) { if (!a) return true; for (long long e = 1; e < M; ++e) if (a[e] != a[0]) return false; return true; };
        const bool ku = all_same(d->k), r0u = all_same(d->r0), rcu = all_same(d->rc);
        s->k_u = (k_arr && M > 0) ? d->k[0] : d->k_uniform;
        s->r0_u = (r0_arr && M > 0) ? d->r0[0] : d->r0_uniform;
        s->rc_u = (rc_arr && M > 0) ? d->rc[0] : d->rc_uniform;
        if (!k_arr) s->k_u = d->k_uniform;
        if (!r0_arr) s->r0_u = d->r0_uniform;
        if (!rc_arr) s->rc_u = d->rc_uniform;
        auto getk = [&](long long e) { return k_arr ? d->k[e] : s->k_u; };
        auto getr0 = [&](long long e) { return r0_arr ? d->r0[e] : s->r0_u; };
        auto getrc = [&](long long e) { return rc_arr ? d->rc[e] : s->rc_u; };
        struct Key { uint64_t a, b, c; bool operator==(const Key &o) const { return a == o.a && b == o.b && c == o.c; } };
        struct KeyHash { size_t operator()(const Key &k) const { return (size_t)(k.a * 0x9E3779B97F4A7C15ull ^ (k.b + 0x7F4A7C15ull) * 0xC2B2AE3D27D4EB4Full ^ (k.c * 0x165667B19E3779F9ull)); } };
        auto bits = [](double v) { uint64_t u; std::memcpy(&u, &v, 8); return u; };
        auto build_table = [&](bool with_rc) -> bool {  // false if more than kMaxTypes distinct entries
            std::unordered_map<Key, int, KeyHash> map;
            stype.assign(M, 0); tab.clear();
            for (long long e = 0; e < M; ++e) {
                Key key{bits(getk(e)), bits(getr0(e)), with_rc ? bits(getrc(e)) : 0};
                auto it = map.find(key);
                if (it == map.end()) {
                    if ((int)map.size() == kMaxTypes) return false;
                    it = map.emplace(key, (int)map.size()).first;
                    tab.push_back(getk(e)); tab.push_back(getr0(e)); tab.push_back(with_rc ? getrc(e) : 0.0);
                }
                stype[e] = (uint8_t)it->second;
            }
            return true;
        };
        if (ku && r0u && rcu) s->pm = PM_UNIFORM;
        else if (build_table(true)) s->pm = PM_TYPED;
        else if (ku && r0u) s->pm = PM_RCF;
        else if (build_table(false)) s->pm = PM_KRT_RCF;
        else s->pm = PM_FULL;
        if (s->pm != PM_TYPED && s->pm != PM_KRT_RCF) { stype.clear(); tab.clear(); }
        s->ntypes = (int)(tab.size() / 3);
    }
    const bool need_typ = s->pm == PM_TYPED || s->pm == PM_KRT_RCF;
    const bool need_rcF = s->pm == PM_RCF || s->pm == PM_KRT_RCF || s->pm == PM_FULL;
    const bool need_krF = s->pm == PM_FULL;
    auto getk = [&](long long e) { return k_arr ? d->k[e] : s->k_u; };
    auto getr0 = [&](long long e) { return r0_arr ? d->r0[e] : s->r0_u; };
    auto getrc = [&](long long e) { return rc_arr ? d->rc[e] : s->rc_u; };

    // ---- particle state ----
    {
        s->T = (N + kTile - 1) / kTile;
        s->Npad = s->T * kTile;                       // the streamed kernel copies whole tiles: pad the tail tile
        const long long Np = s->Npad;
        if (D == 3) {
            const double4 z4 = make_double4(0.0, 0.0, 0.0, 0.0);
            std::vector<double4> hx(Np, z4), hv(Np, z4);
            for (long long c = 0; c < N; ++c) {
                const int32_t p = to_int(c);
                hx[p] = make_double4(d->x[3 * c], d->x[3 * c + 1], d->x[3 * c + 2], 0.0);
                if (d->v) hv[p] = make_double4(d->v[3 * c], d->v[3 * c + 1], d->v[3 * c + 2], 0.0);
            }
            TRY(upload(s, &s->pos3[0], hx));
            s->h_ref3 = hx;
            TRY(dev_alloc(s, &s->pos3[1], (size_t)Np));
            CUDA_TRY(s, cudaMemcpyAsync(s->pos3[1], s->pos3[0], sizeof(double4) * Np, cudaMemcpyDeviceToDevice, s->stream));
            TRY(upload(s, &s->vel3, hv));
            TRY(dev_alloc(s, &s->f3, (size_t)N));
            TRY(dev_alloc(s, &s->fd3, (size_t)N));
            TRY(dev_alloc(s, &s->stage3[0], (size_t)N * 3));
            TRY(dev_alloc(s, &s->stage3[1], (size_t)N * 3));
            CUDA_TRY(s, cudaMemsetAsync(s->f3, 0, sizeof(double4) * N, s->stream));
            CUDA_TRY(s, cudaMemsetAsync(s->fd3, 0, sizeof(double4) * N, s->stream));
            CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        } else {
        std::vector<double2> hx(Np, make_double2(0.0, 0.0)), hv(Np, make_double2(0.0, 0.0));
        for (long long c = 0; c < N; ++c) {
            const int32_t p = to_int(c);
            hx[p] = make_double2(d->x[2 * c], d->x[2 * c + 1]);
            hv[p] = d->v ? make_double2(d->v[2 * c], d->v[2 * c + 1]) : make_double2(0.0, 0.0);
        }
        TRY(upload(s, &s->pos[0], hx));
        s->h_ref2 = hx;
        TRY(dev_alloc(s, &s->pos[1], (size_t)Np));
        CUDA_TRY(s, cudaMemcpyAsync(s->pos[1], s->pos[0], sizeof(double2) * Np, cudaMemcpyDeviceToDevice, s->stream));
        TRY(upload(s, &s->vel, hv));
        TRY(dev_alloc(s, &s->f, (size_t)N));
        TRY(dev_alloc(s, &s->fd, (size_t)N));
        TRY(dev_alloc(s, &s->stage[0], (size_t)N));
        TRY(dev_alloc(s, &s->stage[1], (size_t)N));
        CUDA_TRY(s, cudaMemsetAsync(s->f, 0, sizeof(double2) * N, s->stream));
        CUDA_TRY(s, cudaMemsetAsync(s->fd, 0, sizeof(double2) * N, s->stream));
        }
        s->h_grp.assign(Np, kFree);
        TRY(upload(s, &s->grp, s->h_grp));
        s->h_grp.resize(N);
        if (d->mass) {
            std::vector<double> hm(N);
            for (long long c = 0; c < N; ++c) hm[to_int(c)] = d->mass[c];
            TRY(upload(s, &s->mass, hm));
        }
        if (!s->inv.empty()) TRY(upload(s, &s->d_inv, s->inv));
        TRY(upload(s, &s->d_poff, s->poff));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));  // host vectors go out of scope
    }

    // ---- breakage bookkeeping ----
    TRY(dev_alloc(s, &s->break_step, (size_t)M));
    CUDA_TRY(s, cudaMemsetAsync(s->break_step, 0xFF, sizeof(long long) * std::max<long long>(M, 1), s->stream));  // -1
    TRY(dev_alloc(s, &s->nbroken, (size_t)B));
    CUDA_TRY(s, cudaMemsetAsync(s->nbroken, 0, sizeof(unsigned long long) * B, s->stream));
    TRY(dev_alloc(s, &s->d_broken, (size_t)M));

    // ---- spring layout ----
    if (s->force_mode == LSM_FORCE_GATHER) {
        const long long S = (N + kSlice - 1) / kSlice;
        const long long T = s->T;
        s->nslices = S;
        std::vector<uint32_t> deg(N, 0);
        for (long long e = 0; e < M; ++e) { deg[to_int(d->spring_i[e])]++; deg[to_int(d->spring_j[e])]++; }
        std::vector<uint32_t> off(T * kTileSlices + 1, 0);
        std::vector<TileHdr> hh(T);
        std::memset(hh.data(), 0, sizeof(TileHdr) * T);
        for (long long sl = 0; sl < T * kTileSlices; ++sl) {
            uint32_t w = 0;
            for (long long p = sl * kSlice; p < std::min<long long>(N, (sl + 1) * kSlice); ++p) w = std::max(w, deg[p]);
            if (w > 255) return fail(s, LSM_E_UNSUPPORTED, "particle degree above 255 is not supported by the gather layout; use force_mode = SCATTER");
            const uint64_t nxt = (uint64_t)off[sl] + w;
            if (nxt > 0x07FFFFFFull) return fail(s, LSM_E_UNSUPPORTED, "gather layout too large");
            off[sl + 1] = (uint32_t)nxt;
            TileHdr &h = hh[sl / kTileSlices];
            h.off[sl % kTileSlices] = off[sl];
            h.off[sl % kTileSlices + 1] = off[sl + 1];
            h.w[sl % kTileSlices] = (uint8_t)w;
        }
        s->max_tile_slots = 0;
        for (long long t = 0; t < T; ++t) s->max_tile_slots = std::max(s->max_tile_slots, hh[t].off[kTileSlices] - hh[t].off[0]);
        const size_t E = (size_t)off[T * kTileSlices] * kSlice;
        s->E = (long long)E;
        s->E0 = (long long)off[T * kTileSlices];
        {
            std::vector<uint32_t> tot(2, off[T * kTileSlices]);
            TRY(upload(s, &s->rp_totals, tot));
            CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        }
        std::vector<int32_t> hn(E), hs(E, -1);
        for (long long sl = 0; sl < T * kTileSlices; ++sl)       // padding slots point at their own particle
            for (size_t e = (size_t)off[sl] * kSlice; e < (size_t)off[sl + 1] * kSlice; ++e) hn[e] = (int32_t)(sl * kSlice + (e & 31));
        std::vector<uint8_t> cnt(N, 0);
        auto slot = [&](int32_t p) { const size_t e = ((size_t)off[p >> 5] + cnt[p]) * kSlice + (p & 31); cnt[p]++; return e; };
        for (long long e = 0; e < M; ++e) {  // caller order -> every row is ascending in caller spring id
            const int32_t a = to_int(d->spring_i[e]), b2 = to_int(d->spring_j[e]);
            const size_t ea = slot(a), eb = slot(b2);
            hn[ea] = b2; hs[ea] = (int32_t)e;
            hn[eb] = a; hs[eb] = (int32_t)e;
        }
        TRY(upload(s, &s->hdr, hh));
        TRY(upload(s, &s->nbr, hn));
        bool fits16 = true;
        {   // 16-bit neighbour offsets (neighbour - self) when every one fits: halves the streamed id bytes
            std::vector<int16_t> h16;
            if (fits16) {
                h16.resize(E);
                for (long long sl = 0; sl < T * kTileSlices && fits16; ++sl)
                    for (size_t e = (size_t)off[sl] * kSlice; e < (size_t)off[sl + 1] * kSlice; ++e) {
                        const long long dlt = (long long)hn[e] - (sl * kSlice + (long long)(e & 31));
                        if (dlt < -32768 || dlt > 32767) { fits16 = false; break; }
                        h16[e] = (int16_t)dlt;
                    }
            }
            if (fits16) { TRY(upload(s, &s->nbr16, h16)); CUDA_TRY(s, cudaStreamSynchronize(s->stream)); }
        }
        if (need_typ) { std::vector<uint8_t> ht(E, 0); for (size_t e = 0; e < E; ++e) if (hs[e] >= 0) ht[e] = stype[hs[e]]; TRY(upload(s, &s->typ, ht)); CUDA_TRY(s, cudaStreamSynchronize(s->stream)); }
        if (need_rcF) {
            // 8-bit code of the filter word: base = the smallest word, shift = as few bits as make the spread fit;
            // codes are rounded DOWN (a lower threshold only sends a few more springs to the exact decision)
            uint32_t lo = 0xFFFFFFFFu, hi = 0;
            for (long long e = 0; e < M; ++e) { const uint32_t t = thr_of(getrc(e)); lo = std::min(lo, t); hi = std::max(hi, t); }
            if (M == 0) lo = hi = 0;
            uint32_t shift = 0;
            while (((hi - lo) >> shift) > 0xFFu) ++shift;
            s->thr_base = lo; s->thr_shift = shift;
            std::vector<thr_t> h(E, (thr_t)0xFFu);
            for (size_t e = 0; e < E; ++e) if (hs[e] >= 0) h[e] = (thr_t)((thr_of(getrc(hs[e])) - lo) >> shift);
            TRY(upload(s, &s->thr, h)); CUDA_TRY(s, cudaStreamSynchronize(s->stream));
            std::vector<double> hr(M);
            for (long long e = 0; e < M; ++e) hr[e] = getrc(e);
            TRY(upload(s, &s->rcS, hr)); CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        }
        if (need_krF) {
            std::vector<double> h(E, 0.0);
            for (size_t e = 0; e < E; ++e) if (hs[e] >= 0) h[e] = getk(hs[e]);
            TRY(upload(s, &s->kF, h)); CUDA_TRY(s, cudaStreamSynchronize(s->stream));
            for (size_t e = 0; e < E; ++e) if (hs[e] >= 0) h[e] = getr0(hs[e]);
            TRY(upload(s, &s->r0F, h)); CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        }
        TRY(upload(s, &s->sid, hs));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        // ---- streamed-kernel stage layout: pipeline depth from the largest tile ----
        {
            StageLayout &L = s->L;
            std::memset(&L, 0, sizeof(L));
            auto up = [](int x) { return (x + 127) & ~127; };
            const int cap = (int)s->max_tile_slots;
            int o = 0;
            const int vb = D == 3 ? 32 : 16;   // bytes per position / velocity record
            L.pos = o; o += kTile * vb;
            L.vel = o; o += kTile * vb;
            L.hdr = o; o += 128;
            L.grp = o; o += kTile;
            L.nbr = o; o += up(cap * kSlice * (s->nbr16 ? 2 : 4));
            L.thr = o; if (need_rcF) o += up(cap * kSlice * kThrB);
            L.typ = o; if (need_typ) o += up(cap * kSlice);
            L.kF = o; if (need_krF) o += up(cap * kSlice * 8);
            L.r0F = o; if (need_krF) o += up(cap * kSlice * 8);
            L.bytes = up(o);
            L.first = kStreamHdrBytes + (need_typ ? ((s->ntypes * kTabStride * 8 + 127) & ~127) : 0);
            int dev_smem = 0, n_sm = 0;
            CUDA_TRY(s, cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, d->device));
            CUDA_TRY(s, cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, d->device));
            int ctas_per_sm = kStreamMinB, max_stages = 3;   // 3 stages: within noise of 4, leaves more of the SM for L1 (gathers)
            // big tiles (high degree, 3-D records): fewer resident CTAs per SM until at least two stages fit
            for (;; --ctas_per_sm) {
                const int budget = std::min(dev_smem, (dev_smem + 1024) / ctas_per_sm - 1024) - L.first;   // 1 KB reserved per CTA
                L.stages = std::min<int>(max_stages, budget / std::max(L.bytes, 1));
                if (L.stages >= 2 || ctas_per_sm == 1) break;
            }
            const bool can_stream = L.stages >= 2;
            if (s->gather_variant == 0) s->gather_variant = can_stream ? 2 : 1;
            if (s->gather_variant == 2 && !can_stream) return fail(s, LSM_E_UNSUPPORTED, "gather_variant = streamed: a tile's rows do not fit in shared memory (degree too high); use the direct variant");
            s->stream_smem = L.first + L.stages * L.bytes;
            s->stream_grid = (int)std::min<long long>(T, (long long)ctas_per_sm * n_sm);
            s->stream_ctas_per_sm = ctas_per_sm;
            // step fusion (several time steps per cooperative launch): pays when a step is launch-bound, i.e. the
            // problem is L2-resident; above that the per-step grid barrier costs more than the launch gap it removes.
            int coop = 0;
            CUDA_TRY(s, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, d->device));
            const long long fuse_below = 1 << 18;   // measured: 64^2 5.8 -> 3.6 us per step, 512^2 8.4 -> 8.3, 2.1 M particles 39.1 -> 40.4
            if (s->step_fusion == LSM_FUSION_ON && !(coop && s->gather_variant == 2)) return fail(s, LSM_E_UNSUPPORTED, "step_fusion = ON needs the streamed gather kernel and cooperative launch support");
            s->multi_on = coop && s->gather_variant == 2 && (s->step_fusion == LSM_FUSION_ON || ((s->step_fusion == LSM_FUSION_AUTO || s->step_fusion == LSM_FUSION_RESIDENT) && N <= fuse_below));
            // ---- windowed gathers: the neighbour id ranges of every tile (lsm_window.cuh) ----
            // AUTO: windows up to 2^25 particles.  Measured on B200 (uniform lattices, us per step, windows / global gathers):
            // 4096^2 208 / 234, 1024 x 128^2 244 / 266, config 3 44.9 / 48.9 -- but 6144^2 597 / 495, 8192^2 1068 / 957: there
            // the bulk-copied neighbour ranges miss L2 (hit rate 23 % against 43 %, DRAM reads 4.4 GB against 3.0 GB per step).
            const bool want_win = d->gather_window == LSM_WINDOW_ON || (d->gather_window == LSM_WINDOW_AUTO && N <= (1LL << 25));
            if (D == 2 && s->nbr16 && s->gather_variant == 2 && want_win) {
                std::vector<TileWin> tw(T);
                std::vector<uint16_t> hw(E);
                std::vector<int32_t> ids;
                bool ok = true;
                long long cap = 0;
                for (long long t = 0; t < T && ok; ++t) {
                    const long long p0 = t * kTile, p1 = std::min<long long>(s->Npad, p0 + kTile);
                    const size_t e_lo = (size_t)hh[t].off[0] * kSlice, e_hi = (size_t)hh[t].off[kTileSlices] * kSlice;
                    ids.clear();
                    for (size_t e = e_lo; e < e_hi; ++e) ids.push_back(hn[e]);
                    ids.push_back((int32_t)p0); ids.push_back((int32_t)(p1 - 1));
                    std::sort(ids.begin(), ids.end());
                    ids.erase(std::unique(ids.begin(), ids.end()), ids.end());
                    // ranges: cut where more than 32 ids are skipped (never inside the own particles p0 .. p1-1); if that gives
                    // more than kWinMaxSeg ranges, the smallest gaps are bridged
                    TileWin &w = tw[t];
                    std::memset(&w, 0, sizeof(w));
                    std::vector<std::pair<long long, size_t>> cuts;      // (gap, index of the first id after the cut)
                    for (size_t q = 1; q < ids.size(); ++q) {
                        const bool own_gap = ids[q - 1] >= p0 && ids[q] < p1;
                        if (ids[q] - ids[q - 1] > 32 && !own_gap) cuts.push_back({(long long)ids[q] - ids[q - 1], q});
                    }
                    if ((int)cuts.size() > kWinMaxSeg - 1) {
                        std::sort(cuts.begin(), cuts.end(), [](const auto &a, const auto &b) { return a.first > b.first; });
                        cuts.resize(kWinMaxSeg - 1);
                    }
                    std::sort(cuts.begin(), cuts.end(), [](const auto &a, const auto &b) { return a.second < b.second; });
                    int nseg = 0;
                    long long tot = 0;
                    size_t first = 0;
                    for (size_t c = 0; c <= cuts.size(); ++c) {
                        const size_t last = (c < cuts.size() ? cuts[c].second : ids.size()) - 1;
                        const long long len = (long long)ids[last] - ids[first] + 1;
                        if (len > 65535) { ok = false; break; }
                        w.start[nseg] = ids[first]; w.len[nseg] = (uint16_t)len; tot += len; ++nseg;
                        first = last + 1;
                    }
                    if (tot > 4096) ok = false;                          // a window this wide would not leave two pipeline stages
                    if (!ok || tot > 65535) { ok = false; break; }
                    cap = std::max(cap, tot);
                    auto index_of = [&](int32_t id) { long long o = 0; for (int q = 0; q < nseg; ++q) { if (id >= w.start[q] && id < w.start[q] + (int32_t)w.len[q]) return (uint16_t)(o + id - w.start[q]); o += w.len[q]; } return (uint16_t)0; };
                    w.own_base = index_of((int32_t)p0);
                    uint16_t ob = w.own_base;
                    std::memcpy(hh[t].pad, &ob, 2);
                    for (size_t e = e_lo; e < e_hi; ++e) hw[e] = index_of(hn[e]);
                }
                if (d->gather_window == LSM_WINDOW_ON && !ok) return fail(s, LSM_E_UNSUPPORTED, "gather_window = ON: a tile's neighbours do not form <= 4 short id ranges (numbering not banded)");
                if (ok) {
                    StageLayout LW = s->L;
                    const int extra = ((int)((cap * 16 + 127) & ~127LL)) - kTile * 16;      // the window replaces the own-position block
                    LW.vel += extra; LW.hdr += extra; LW.grp += extra; LW.nbr += extra; LW.thr += extra; LW.typ += extra; LW.kF += extra; LW.r0F += extra;
                    LW.bytes += extra;
                    int ctas = s->stream_ctas_per_sm;
                    for (;; --ctas) {
                        const int budget = std::min(dev_smem, (dev_smem + 1024) / ctas - 1024) - LW.first;
                        LW.stages = std::min<int>(max_stages, budget / std::max(LW.bytes, 1));
                        if (LW.stages >= 2 || ctas == 1) break;
                    }
                    if (LW.stages >= 2) {
                        s->win_on = 1; s->win_cap = (int)cap; s->LW = LW;
                        s->win_smem = LW.first + LW.stages * LW.bytes;
                        s->win_grid = (int)std::min<long long>(T, (long long)ctas * n_sm);
                        CUDA_TRY(s, cudaMemcpyAsync(s->hdr, hh.data(), sizeof(TileHdr) * T, cudaMemcpyHostToDevice, s->stream));   // own_base in the pad bytes
                        TRY(upload(s, &s->d_win, tw));
                        TRY(upload(s, &s->widx, hw));
                        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
                        // cooperative multi-step launches: tiles resident in the stages, windows re-fetched after the grid barrier
                        // (measured: 512^2 6.67 against 7.07 us per step with L2 gathers; with one tile per CTA the extra bulk-copy round
                        //  trip behind the barrier costs more than the gathers it replaces: 46k particles 3.67 against 3.29 us)
                        if (s->multi_on && T > s->win_grid && (T + s->win_grid - 1) / s->win_grid <= LW.stages) s->coopwin_on = 1;
                    } else if (d->gather_window == LSM_WINDOW_ON) return fail(s, LSM_E_UNSUPPORTED, "gather_window = ON: the windows do not fit two pipeline stages");
                }
            } else if (d->gather_window == LSM_WINDOW_ON) return fail(s, LSM_E_UNSUPPORTED, "gather_window = ON needs dim = 2, the streamed gather kernel and 16-bit neighbour offsets");
            // cluster-resident stepping: units (specimens) small enough for one thread-block cluster's shared memory
            const bool want_res = s->step_fusion == LSM_FUSION_RESIDENT || s->step_fusion == LSM_FUSION_AUTO;
            if (want_res && D == 2 && s->nbr16 && s->gather_variant == 2 && N <= 0x7FFFFFFF) {
                std::vector<int32_t> nbmin(N), nbmax(N);
                for (long long p = 0; p < N; ++p) {
                    int32_t lo = (int32_t)p, hi = (int32_t)p;
                    for (uint32_t q = off[p >> 5]; q < off[(p >> 5) + 1]; ++q) { const int32_t nb = hn[(size_t)q * kSlice + (p & 31)]; lo = std::min(lo, nb); hi = std::max(hi, nb); }
                    nbmin[p] = lo; nbmax[p] = hi;
                }
                const int budget = dev_smem - 2048;            // static shared memory (the CTA descriptor) + reserve
                ResPlan best;
                for (int C = 1; C <= kResMaxCluster; C *= 2) {
                    if (s->cluster_size > 0 && C != s->cluster_size) continue;
                    ResPlan R = plan_resident(s, C, nbmin, nbmax, off, budget);
                    if (!R.ok) continue;
                    // a plan counts only if this device can place such a cluster (sizes above 8 are non-portable, each CTA
                    // asks for most of an SM's shared memory); otherwise the next size, or the other schedules, take over
                    R.active = resident_clusters(s, C, R.L.bytes);
                    if (R.active < 1) continue;
                    if (!best.ok) { best = std::move(R); if (s->cluster_size > 0) break; continue; }
                    // a single (or a few) small units: more CTAs per unit while the GPU is not full and each keeps >= 8 slices
                    if ((long long)B * C <= n_sm && R.L.sl_cap >= 8) best = std::move(R); else break;
                }
                // AUTO: a cluster uses at most 16 SMs, so one mid-size lattice is better off on the whole GPU with the
                // cooperative multi-step launch (measured: 46k particles 3.3 us per step there, 6.0 us on one cluster);
                // resident pays when the clusters fill the GPU, or when each warp has about one slice per step
                if (best.ok && s->step_fusion == LSM_FUSION_AUTO && !((long long)B * best.C * 2 >= n_sm || best.L.sl_cap <= 16)) best.ok = false;
                if (best.ok) {
                    s->res_on = 1; s->res_cluster = best.C; s->res_grid = B * best.C; s->RL = best.L; s->res_active_clusters = best.active;
                    TRY(upload(s, &s->res_desc, best.desc));
                    TRY(upload(s, &s->res_order, best.order));
                    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
                    s->multi_on = 0;                               // the cluster barrier replaces the grid barrier
                }
            }
            if (s->step_fusion == LSM_FUSION_RESIDENT && !s->res_on) return fail(s, LSM_E_UNSUPPORTED, "step_fusion = RESIDENT: needs dim = 2, the streamed gather kernel, 16-bit neighbour offsets (a banded numbering), specimens that start on multiples of 32 particles and fit one cluster's shared memory, CTAs whose ghost exchange is mutual, and a device that can place such a cluster");
            if (s->multi_on) {
                TRY(dev_alloc(s, &s->gbar, 1));
                CUDA_TRY(s, cudaMemsetAsync(s->gbar, 0, sizeof(unsigned long long), s->stream));
            }
        }
    } else if (s->force_mode == LSM_FORCE_SCATTER) {
        if (s->exact) return fail(s, LSM_E_UNSUPPORTED, "exact arithmetic needs force_mode = GATHER (atomic summation order is not fixed)");
        // spring list in internal numbering, sorted by (lower endpoint, upper endpoint) for gather / atomic locality
        std::vector<int32_t> order(M);
        for (long long e = 0; e < M; ++e) order[e] = (int32_t)e;
        std::vector<int32_t> a(M), b2(M);
        for (long long e = 0; e < M; ++e) { int32_t i = to_int(d->spring_i[e]), j = to_int(d->spring_j[e]); a[e] = std::min(i, j); b2[e] = std::max(i, j); }
        std::sort(order.begin(), order.end(), [&](int32_t x, int32_t y) { return a[x] != a[y] ? a[x] < a[y] : (b2[x] != b2[y] ? b2[x] < b2[y] : x < y); });
        std::vector<int32_t> hi(M), hj(M), hs(M);
        for (long long q = 0; q < M; ++q) { const int32_t e = order[q]; hi[q] = to_int(d->spring_i[e]); hj[q] = to_int(d->spring_j[e]); hs[q] = e; }
        if (s->scatter_variant != 0) {   // aggregated variants: (lower endpoint, upper endpoint); f_lo += g d, f_hi -= g d with d = x_hi - x_lo
            for (long long q = 0; q < M; ++q) if (hi[q] > hj[q]) std::swap(hi[q], hj[q]);
            std::vector<int32_t> own(N + 1, 0), jlo(N + 1, 0), jli;
            for (long long q = 0; q < M; ++q) own[hi[q] + 1]++;
            for (long long p = 0; p < N; ++p) own[p + 1] += own[p];
            const long long ntile = (N + kScatterTile - 1) / kScatterTile;
            std::vector<int32_t> toff(ntile + 1, 0);
            for (long long t = 0; t <= ntile; ++t) toff[t] = own[std::min<long long>(N, t * kScatterTile)];
            long long cap = 0;
            for (long long t = 0; t < ntile; ++t) cap = std::max<long long>(cap, toff[t + 1] - toff[t]);
            // springs a particle is the UPPER endpoint of, lower endpoint in the same tile (the others spill with a RED)
            for (long long q = 0; q < M; ++q) if (hi[q] / kScatterTile == hj[q] / kScatterTile) jlo[hj[q] + 1]++;
            for (long long p = 0; p < N; ++p) jlo[p + 1] += jlo[p];
            jli.resize(std::max<long long>(jlo[N], 1));
            { std::vector<int32_t> fill(jlo.begin(), jlo.end() - 1); for (long long q = 0; q < M; ++q) if (hi[q] / kScatterTile == hj[q] / kScatterTile) jli[fill[hj[q]]++] = (int32_t)q; }
            s->scatter_tiles = (int)ntile; s->scatter_tile_smem = (int)(cap * 16);
            if (s->scatter_variant == 2 && s->scatter_tile_smem > 200 * 1024) return fail(s, LSM_E_UNSUPPORTED, "force_mode = SCATTER_TILE: a tile's springs do not fit in shared memory (degree too high)");
            TRY(upload(s, &s->s_own_off, own)); TRY(upload(s, &s->s_jl_off, jlo)); TRY(upload(s, &s->s_jl_idx, jli)); TRY(upload(s, &s->s_tile_off, toff));
            CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        }
        s->Ms = M; s->E = M;
        TRY(upload(s, &s->ssi, hi)); TRY(upload(s, &s->ssj, hj)); TRY(upload(s, &s->ssid, hs));
        if (need_typ) { std::vector<uint8_t> ht(M); for (long long q = 0; q < M; ++q) ht[q] = stype[hs[q]]; TRY(upload(s, &s->typ, ht)); CUDA_TRY(s, cudaStreamSynchronize(s->stream)); }
        if (need_rcF) { std::vector<double> h(M); for (long long q = 0; q < M; ++q) h[q] = getrc(hs[q]); TRY(upload(s, &s->rcF, h)); CUDA_TRY(s, cudaStreamSynchronize(s->stream)); }
        if (need_krF) {
            std::vector<double> h(M);
            for (long long q = 0; q < M; ++q) h[q] = getk(hs[q]);
            TRY(upload(s, &s->kF, h)); CUDA_TRY(s, cudaStreamSynchronize(s->stream));
            for (long long q = 0; q < M; ++q) h[q] = getr0(hs[q]);
            TRY(upload(s, &s->r0F, h)); CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        }
        TRY(dev_alloc(s, &s->sUs, (size_t)M));
        // specimen segments of the sorted list (sorted by lower endpoint, specimens are contiguous id ranges)
        std::vector<long long> sl(B + 1, 0);
        { int b = 0; for (long long q = 0; q < M; ++q) { while (std::min(hi[q], hj[q]) >= s->poff[b + 1]) { ++b; sl[b] = q; } } for (int bb = b + 1; bb <= B; ++bb) sl[bb] = M; }
        TRY(upload(s, &s->d_soff_list, sl));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    } else {
        return fail(s, LSM_E_INVALID, "bad force_mode");
    }
    if (!tab.empty()) {
        if (s->force_mode == LSM_FORCE_GATHER) {   // gather kernels: kTabStride doubles per type (k, k*r0, filter word, r0, rc)
            std::vector<double> t4(tab.size() / 3 * kTabStride, 0.0);
            for (size_t t = 0; t < tab.size() / 3; ++t) {
                const double k = tab[3 * t], r0 = tab[3 * t + 1], rc = tab[3 * t + 2];
                double *q = &t4[kTabStride * t];
                q[0] = k; q[1] = k * r0; q[3] = r0; q[4] = rc;
                const uint64_t w = thr_of(rc);
                std::memcpy(&q[2], &w, 8);
            }
            tab.swap(t4);
        }
        TRY(upload(s, &s->tab, tab)); CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    }

    // ---- reductions: chunk table, scratch, history ring ----
    {
        std::vector<long long> lo, hi;
        std::vector<int> sco(B + 1, 0);
        for (int b = 0; b < B; ++b) {
            for (long long p = s->poff[b]; p < s->poff[b + 1]; p += kChunk) { lo.push_back(p); hi.push_back(std::min(p + kChunk, s->poff[b + 1])); }
            sco[b + 1] = (int)lo.size();
        }
        s->nchunks = (long long)lo.size();
        TRY(upload(s, &s->chunk_lo, lo)); TRY(upload(s, &s->chunk_hi, hi)); TRY(upload(s, &s->spec_chunk_off, sco));
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        TRY(dev_alloc(s, &s->part, (size_t)s->nchunks * 2));
        TRY(dev_alloc(s, &s->sU, (size_t)N)); TRY(dev_alloc(s, &s->sKE, (size_t)N));
        TRY(dev_alloc(s, &s->flags, 2));               // [0] sticky device-side error bits, [1] scratch of the input validation
        CUDA_TRY(s, cudaMemsetAsync(s->flags, 0, 2 * sizeof(int), s->stream));
        TRY(dev_alloc(s, &s->cur_U, (size_t)B)); TRY(dev_alloc(s, &s->cur_KE, (size_t)B));
        const size_t cap = (size_t)s->hist_cap;
        TRY(dev_alloc(s, &s->hist_step, cap)); TRY(dev_alloc(s, &s->hist_nb, cap * B));
        TRY(dev_alloc(s, &s->hist_R, cap * B * kMaxGroups * D));
        TRY(dev_alloc(s, &s->hist_U, cap * B)); TRY(dev_alloc(s, &s->hist_KE, cap * B));
    }
    s->step = 0;
    TRY(eval_initial(s));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    return LSM_OK;
}

lsm_status lsm_create(const lsm_desc *d, lsm_sim **out) {
    if (out) *out = nullptr;
    if (!d || !out) return fail(nullptr, LSM_E_INVALID, "desc / out is NULL");
    if (d->struct_size != sizeof(lsm_desc)) return fail(nullptr, LSM_E_INVALID, "lsm_desc.struct_size does not match this library (ABI mismatch)");
    if (d->dim != 2 && d->dim != 3) return fail(nullptr, LSM_E_INVALID, "dim must be 2 or 3");
    if (d->dim == 3 && (d->force_mode == LSM_FORCE_SCATTER || d->force_mode == LSM_FORCE_SCATTER_WARP || d->force_mode == LSM_FORCE_SCATTER_TILE)) return fail(nullptr, LSM_E_UNSUPPORTED, "dim = 3 has no scatter path");
    if (d->n_particles < 1 || d->n_springs < 0 || d->n_particles >= 2147483647LL || d->n_springs >= 2147483647LL) return fail(nullptr, LSM_E_INVALID, "need 1 <= N < 2^31-1 and 0 <= M < 2^31-1");
    if (d->n_batch < 1 || !d->x) return fail(nullptr, LSM_E_INVALID, "n_batch < 1 or x is NULL");
    if (!(d->dt > 0.0) || !(d->gamma >= 0.0) || !std::isfinite(d->dt) || !std::isfinite(d->gamma)) return fail(nullptr, LSM_E_INVALID, "need dt > 0 and gamma >= 0");
    if (d->sample_every < 0 || d->compact_every < 0 || d->history_capacity < 0) return fail(nullptr, LSM_E_INVALID, "negative sample_every / compact_every / history_capacity");
    if (d->reorder < LSM_REORDER_NONE || d->reorder > LSM_REORDER_BLOCKED) return fail(nullptr, LSM_E_INVALID, "bad reorder");
    if (d->reorder == LSM_REORDER_BLOCKED && d->dim != 2) return fail(nullptr, LSM_E_UNSUPPORTED, "reorder = BLOCKED is 2-D only");
    if (d->force_mode < 0 || d->force_mode > LSM_FORCE_SCATTER_TILE) return fail(nullptr, LSM_E_INVALID, "bad force_mode");
    if (d->gather_variant < 0 || d->gather_variant > 2) return fail(nullptr, LSM_E_INVALID, "bad gather_variant");
    if (d->gather_window < 0 || d->gather_window > 2) return fail(nullptr, LSM_E_INVALID, "bad gather_window");
    if (d->step_fusion < 0 || d->step_fusion > 3) return fail(nullptr, LSM_E_INVALID, "bad step_fusion");
    if (d->cluster_size != 0 && d->cluster_size != 1 && d->cluster_size != 2 && d->cluster_size != 4 && d->cluster_size != 8 && d->cluster_size != 16) return fail(nullptr, LSM_E_INVALID, "cluster_size must be 0 (auto), 1, 2, 4, 8 or 16");
    if ((d->alloc == nullptr) != (d->free_ == nullptr)) return fail(nullptr, LSM_E_INVALID, "alloc and free_ must be given together");
    lsm_sim *s = new (std::nothrow) lsm_sim();
    if (!s) return fail(nullptr, LSM_E_NOMEM, "out of host memory");
    lsm_status st;
    try { st = create_impl(d, s); }
    catch (const std::bad_alloc &) { st = fail(s, LSM_E_NOMEM, "out of host memory while building the layout"); }
    if (st != LSM_OK) { g_create_error = s->err; lsm_destroy(s); return st; }
    *out = s;
    return LSM_OK;
}

#define CHECK_SIM(s)                               \
    if (!(s)) return LSM_E_INVALID;                \
    if ((s)->sticky != LSM_OK) return (s)->sticky; \
    DeviceScope _device_scope((s)->device)

lsm_status lsm_set_boundary(lsm_sim *s, int32_t gi, const int32_t *ids, int64_t n, int32_t mode, const double *du) {
    CHECK_SIM(s);
    if (gi < 0 || gi >= kMaxGroups) { s->err = "group id out of range"; return LSM_E_RANGE; }
    if (n < 0 || (n > 0 && !ids) || (mode != LSM_FIXED && mode != LSM_MOVE)) { s->err = "bad arguments"; return LSM_E_INVALID; }
    if (mode == LSM_MOVE && (!du || !std::isfinite(du[0]) || !std::isfinite(du[1]) || (s->dim == 3 && !std::isfinite(du[2])))) { s->err = "MOVE needs a finite disp_per_step"; return LSM_E_INVALID; }
    Group &g = s->groups[gi];
    std::vector<int32_t> nid((size_t)n);
    for (long long q = 0; q < n; ++q) {
        if (ids[q] < 0 || ids[q] >= s->N) { s->err = "boundary particle id out of range"; return LSM_E_RANGE; }
        nid[q] = s->inv.empty() ? ids[q] : s->inv[ids[q]];
        const uint8_t cg = s->h_grp[nid[q]];
        if (cg != kFree && cg != gi) { s->err = "particle already belongs to another boundary group"; return LSM_E_RANGE; }
    }
    std::sort(nid.begin(), nid.end());
    if (std::adjacent_find(nid.begin(), nid.end()) != nid.end()) { s->err = "duplicate particle id in the group"; return LSM_E_RANGE; }
    // release the old members: free again, carrying the kinematic velocity du/dt (Q6)
    if (g.set && !g.ids.empty()) {
        if (s->dim == 3) k3_group_release<<<grid_for((long long)g.ids.size()), kBlock, 0, s->stream>>>(g.d_ids, (long long)g.ids.size(), s->grp, s->vel3, g.du[0] / s->dt, g.du[1] / s->dt, g.du[2] / s->dt, s->sKE, s->mass, s->mass_u);
        else k_group_release<<<grid_for((long long)g.ids.size()), kBlock, 0, s->stream>>>(g.d_ids, (long long)g.ids.size(), s->grp, s->vel, g.du[0] / s->dt, g.du[1] / s->dt, s->sKE, s->mass, s->mass_u);
        s->kernels_launched += 1;
        for (int32_t p : g.ids) s->h_grp[p] = kFree;
    }
    if (g.d_ids || g.d_seg) {   // the group's previous device lists: nothing enqueued may still read them
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
        dev_free(s, g.d_ids); dev_free(s, g.d_seg);
        g.d_ids = nullptr; g.d_seg = nullptr;
    }
    g.set = true; g.mode = mode; g.n0 = s->step;
    g.du[0] = mode == LSM_MOVE ? du[0] : 0.0; g.du[1] = mode == LSM_MOVE ? du[1] : 0.0;
    g.du[2] = (mode == LSM_MOVE && s->dim == 3) ? du[2] : 0.0;
    g.ids = nid;
    for (int32_t p : nid) s->h_grp[p] = (uint8_t)gi;
    std::vector<long long> seg(s->B + 1, 0);
    { int b = 0; for (size_t q = 0; q < nid.size(); ++q) { while (nid[q] >= s->poff[b + 1]) { ++b; seg[b] = (long long)q; } } for (int bb = b + 1; bb <= s->B; ++bb) seg[bb] = (long long)nid.size(); }
    TRY(upload(s, &g.d_ids, nid));
    TRY(upload(s, &g.d_seg, seg));
    if (n > 0) {
        if (s->dim == 3) k3_group_assign<<<grid_for(n), kBlock, 0, s->stream>>>(g.d_ids, n, s->grp, s->vel3, s->pos3[s->cur], (uint8_t)gi, s->sKE);
        else k_group_assign<<<grid_for(n), kBlock, 0, s->stream>>>(g.d_ids, n, s->grp, s->vel, s->pos[s->cur], (uint8_t)gi, s->sKE);
        s->kernels_launched += 1;
    }
    CUDA_TRY(s, cudaGetLastError());
    // Membership and origins change, nothing else (R3): positions are untouched, so the spring forces f and the
    // held total force fd = f - gamma v of the last force evaluation stay what they were -- fd still feeds the next first
    // half kick of every free particle (Q7) -- and only the members' kinetic-energy terms were adjusted above.
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));   // nid / seg go out of scope
    return LSM_OK;
}

// Enqueue one lsm_step call: START, (n-1) fused MID steps, END.
lsm_status lsm_step(lsm_sim *s, int64_t n_steps) {
    CHECK_SIM(s);
    if (n_steps < 0) { s->err = "n_steps < 0"; return LSM_E_INVALID; }
    if (n_steps == 0) return LSM_OK;
    const bool gather = s->force_mode == LSM_FORCE_GATHER;
    long long done = 0;
    while (done < n_steps) {
        // split the call at compaction boundaries
        long long seg = n_steps - done;
        if (s->compact_every > 0) seg = std::min<long long>(seg, s->compact_every - (s->step - s->last_compact_step) > 0 ? s->compact_every - (s->step - s->last_compact_step) : 1);
        // START: first half kick + drift from the completed state
        {
            if (s->dim == 3) {
                const Step3Params P3 = step_params3(s, s->step, V_MID);
                if (s->exact) k3_start<true><<<grid_for(s->N), kBlock, 0, s->stream>>>(P3);
                else k3_start<false><<<grid_for(s->N), kBlock, 0, s->stream>>>(P3);
            } else {
                StepParams P = step_params(s, s->step);
                if (s->exact) k_start<true><<<grid_for(s->N), kBlock, 0, s->stream>>>(P);
                else k_start<false><<<grid_for(s->N), kBlock, 0, s->stream>>>(P);
            }
            s->kernels_launched += 1;
            if (gather) s->cur ^= 1;
            else { k_zero_f<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->f, s->N); s->kernels_launched += 1; }
        }
        for (long long i = 1; i <= seg; ++i) {
            const long long m = s->step + i;  // the step this force evaluation completes
            const bool last = i == seg;
            const bool samp = is_sample_step(s, m);
            const Variant v = last ? V_END : (samp ? V_MID_SAMPLE : V_MID);
            if (gather && s->res_on && v == V_MID) {     // the run of plain MID steps that starts here, resident in the clusters
                long long run = 1;
                while (i + run < seg && !is_sample_step(s, m + run) && run < 65536) ++run;
                if (run >= 2) {
                    CUDA_TRY(s, launch_resident(s, m, (int)run));
                    s->kernels_launched += 1;
                    i += run - 1;
                    continue;
                }
            }
            if (gather && s->multi_on && v == V_MID) {   // fuse the run of plain MID steps that starts here into one launch
                long long run = 1;
                while (i + run < seg && !is_sample_step(s, m + run) && run < s->multi_max) ++run;
                if (run >= 2 && s->coopwin_on) {
                    StepParams P = step_params(s, m);
                    CoopWinParams Q;
                    Q.win = s->d_win; Q.widx = s->widx; Q.gbar = s->gbar; Q.gbar_base = s->gbar_base;
                    Q.pos_a = s->pos[s->cur]; Q.pos_b = s->pos[s->cur ^ 1]; Q.nsteps = (int)run;
                    CUDA_TRY(s, s->exact ? launch_coopwin_pm<true>(s, P, Q) : launch_coopwin_pm<false>(s, P, Q));
                    s->gbar_base += (unsigned long long)(run - 1) * (unsigned long long)s->win_grid;
                    s->kernels_launched += 1;
                    if (run & 1) s->cur ^= 1;
                    i += run - 1;
                    continue;
                }
                if (run >= 2) {
                    StepParams P = step_params(s, m);
                    MultiParams Mp;
                    Mp.nsteps = (int)run; Mp.gbar = s->gbar; Mp.gbar_base = s->gbar_base;
                    if (s->dim == 3) { Mp.pos_a = reinterpret_cast<double2 *>(s->pos3[s->cur]); Mp.pos_b = reinterpret_cast<double2 *>(s->pos3[s->cur ^ 1]); }
                    else { Mp.pos_a = s->pos[s->cur]; Mp.pos_b = s->pos[s->cur ^ 1]; }
                    Mp.resident = (s->T + s->stream_grid - 1) / s->stream_grid <= s->L.stages;
                    CUDA_TRY(s, s->exact ? launch_stream_multi_pm<true>(s, P, Mp) : launch_stream_multi_pm<false>(s, P, Mp));
                    s->gbar_base += (unsigned long long)(run - 1) * (unsigned long long)s->stream_grid;
                    s->kernels_launched += 1;
                    if (run & 1) s->cur ^= 1;
                    i += run - 1;
                    continue;
                }
            }
            StepParams P = step_params(s, m);
            if (gather) {
                launch_gather(s, P, v);
                if (!last) s->cur ^= 1;
            } else {
                launch_scatter_force(s, P, samp || last);
                launch_integrate(s, P, v);
            }
            if (samp) record_sample(s, m);
            if (!gather && samp && !last) { k_zero_f<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->f, s->N); s->kernels_launched += 1; }
        }
        s->step += seg;
        done += seg;
        CUDA_TRY(s, cudaGetLastError());
        if (s->compact_every > 0 && s->step - s->last_compact_step >= s->compact_every) TRY(do_compact(s));
    }
    return LSM_OK;
}

lsm_status lsm_compact(lsm_sim *s) {
    CHECK_SIM(s);
    return do_compact(s);
}

static lsm_status check_flags(lsm_sim *s) {
    int fl = 0;
    CUDA_TRY(s, cudaMemcpyAsync(&fl, s->flags, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    if (fl & 1) return fail(s, LSM_E_STATE, "non-finite energy detected on the device: the simulation blew up");
    return LSM_OK;
}

lsm_status lsm_sync(lsm_sim *s) {
    CHECK_SIM(s);
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    return LSM_OK;
}

lsm_status lsm_write_state(lsm_sim *s, const double *x, const double *v) {
    CHECK_SIM(s);
    if (!x) { s->err = "x is NULL"; return LSM_E_INVALID; }
    // stage the caller's arrays, validate them on the device, and only then touch the state
    double *sx = s->dim == 3 ? s->stage3[0] : reinterpret_cast<double *>(s->stage[0]);
    double *sv = s->dim == 3 ? s->stage3[1] : reinterpret_cast<double *>(s->stage[1]);
    const long long n = (long long)s->dim * s->N;
    CUDA_TRY(s, cudaMemcpyAsync(sx, x, sizeof(double) * n, cudaMemcpyHostToDevice, s->stream));
    if (v) CUDA_TRY(s, cudaMemcpyAsync(sv, v, sizeof(double) * n, cudaMemcpyHostToDevice, s->stream));
    CUDA_TRY(s, cudaMemsetAsync(s->flags + 1, 0, sizeof(int), s->stream));
    k_check_finite<<<(unsigned)std::min<long long>(2048, (n + kBlock - 1) / kBlock), kBlock, 0, s->stream>>>(sx, v ? sv : nullptr, n, s->flags + 1);
    s->kernels_launched += 1;
    int bad = 0;
    CUDA_TRY(s, cudaMemcpyAsync(&bad, s->flags + 1, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));   // x / v are borrowed for the duration of the call only (lsm.h): consumed here
    if (bad) { s->err = "non-finite position / velocity"; return LSM_E_NONFINITE; }
    if (s->dim == 3) k3_from_caller<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->stage3[0], v ? s->stage3[1] : nullptr, s->pos3[s->cur], s->vel3, s->d_inv, s->N, s->grp);
    else k_from_caller<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->stage[0], v ? s->stage[1] : nullptr, s->pos[s->cur], s->vel, s->d_inv, s->N, s->grp);
    s->kernels_launched += 1;
    for (int g = 0; g < kMaxGroups; ++g) s->groups[g].n0 = s->step;
    TRY(eval_initial(s));
    return LSM_OK;
}

lsm_status lsm_read_state(lsm_sim *s, double *x, double *v) {
    CHECK_SIM(s);
    if (s->dim == 3) {
        const GroupTab3 g3 = group_tab3(s);
        if (x) {
            k3_to_caller<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->pos3[s->cur], s->stage3[0], s->d_inv, s->N, s->grp, g3, s->dt, 0);
            CUDA_TRY(s, cudaMemcpyAsync(x, s->stage3[0], sizeof(double) * 3 * s->N, cudaMemcpyDeviceToHost, s->stream));
            s->kernels_launched += 1;
        }
        if (v) {
            k3_to_caller<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->vel3, s->stage3[1], s->d_inv, s->N, s->grp, g3, s->dt, 1);
            CUDA_TRY(s, cudaMemcpyAsync(v, s->stage3[1], sizeof(double) * 3 * s->N, cudaMemcpyDeviceToHost, s->stream));
            s->kernels_launched += 1;
        }
        return check_flags(s);
    }
    const GroupTab g = group_tab(s);
    if (x) {
        k_to_caller<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->pos[s->cur], s->stage[0], s->d_inv, s->N, s->grp, g, s->dt, 0);
        CUDA_TRY(s, cudaMemcpyAsync(x, s->stage[0], sizeof(double2) * s->N, cudaMemcpyDeviceToHost, s->stream));
        s->kernels_launched += 1;
    }
    if (v) {
        k_to_caller<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->vel, s->stage[1], s->d_inv, s->N, s->grp, g, s->dt, 1);
        CUDA_TRY(s, cudaMemcpyAsync(v, s->stage[1], sizeof(double2) * s->N, cudaMemcpyDeviceToHost, s->stream));
        s->kernels_launched += 1;
    }
    return check_flags(s);
}

lsm_status lsm_read_forces(lsm_sim *s, double *f) {
    CHECK_SIM(s);
    if (!f) { s->err = "f is NULL"; return LSM_E_INVALID; }
    if (s->dim == 3) {
        k3_to_caller<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->f3, s->stage3[0], s->d_inv, s->N, s->grp, group_tab3(s), s->dt, 0);
        s->kernels_launched += 1;
        CUDA_TRY(s, cudaMemcpyAsync(f, s->stage3[0], sizeof(double) * 3 * s->N, cudaMemcpyDeviceToHost, s->stream));
        return check_flags(s);
    }
    k_to_caller<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->f, s->stage[0], s->d_inv, s->N, s->grp, group_tab(s), s->dt, 0);
    s->kernels_launched += 1;
    CUDA_TRY(s, cudaMemcpyAsync(f, s->stage[0], sizeof(double2) * s->N, cudaMemcpyDeviceToHost, s->stream));
    return check_flags(s);
}

lsm_status lsm_read_virial(lsm_sim *s, double *S) {
    CHECK_SIM(s);
    if (!S) { s->err = "S is NULL"; return LSM_E_INVALID; }
    if (s->force_mode != LSM_FORCE_GATHER) { s->err = "lsm_read_virial needs the gather layout"; return LSM_E_UNSUPPORTED; }
    if (!s->virial) TRY(dev_alloc(s, &s->virial, (size_t)s->N * (s->dim == 3 ? 6 : 3)));
    if (s->dim == 3) {
        Virial3Params V;
        std::memset(&V, 0, sizeof(V));
        const StepParams P = step_params(s, s->step);
        V.pos = s->pos3[s->cur]; V.vel = s->vel3; V.grp = s->grp; V.mass = s->mass; V.mass_u = s->mass_u; V.dt = s->dt;
        V.hdr = s->hdr; V.nbr = s->nbr; V.sp = P.sp; V.pm = s->pm; V.inv = s->d_inv; V.N = s->N; V.g = group_tab3(s); V.out = s->virial;
        k3_virial<<<grid_for(s->N), kBlock, 0, s->stream>>>(V);
        s->kernels_launched += 1;
        CUDA_TRY(s, cudaGetLastError());
        CUDA_TRY(s, cudaMemcpyAsync(S, s->virial, sizeof(double) * 6 * s->N, cudaMemcpyDeviceToHost, s->stream));
        return check_flags(s);
    }
    VirialParams V;
    std::memset(&V, 0, sizeof(V));
    const StepParams P = step_params(s, s->step);
    V.pos = s->pos[s->cur]; V.vel = s->vel; V.grp = s->grp; V.mass = s->mass; V.mass_u = s->mass_u; V.dt = s->dt;
    V.hdr = s->hdr; V.nbr = s->nbr; V.sp = P.sp; V.pm = s->pm; V.inv = s->d_inv; V.N = s->N; V.g = P.g; V.out = s->virial;
    k_virial<<<grid_for(s->N), kBlock, 0, s->stream>>>(V);
    s->kernels_launched += 1;
    CUDA_TRY(s, cudaGetLastError());
    CUDA_TRY(s, cudaMemcpyAsync(S, s->virial, sizeof(double) * 3 * s->N, cudaMemcpyDeviceToHost, s->stream));
    return check_flags(s);
}

lsm_status lsm_read_strain(lsm_sim *s, double *E, uint8_t *ok) {
    CHECK_SIM(s);
    if (!E) { s->err = "E is NULL"; return LSM_E_INVALID; }
    if (s->force_mode != LSM_FORCE_GATHER) { s->err = "lsm_read_strain needs the gather layout"; return LSM_E_UNSUPPORTED; }
    const int C = s->dim == 3 ? 6 : 3;
    if (!s->strain) {
        TRY(dev_alloc(s, &s->strain, (size_t)s->N * C));
        TRY(dev_alloc(s, &s->strain_ok, (size_t)s->N));
        if (s->dim == 3) TRY(upload(s, &s->ref3, s->h_ref3)); else TRY(upload(s, &s->ref2, s->h_ref2));
    }
    if (s->dim == 3) {
        StrainParams<double4> S;
        S.pos = s->pos3[s->cur]; S.ref = s->ref3; S.hdr = s->hdr; S.nbr = s->nbr; S.inv = s->d_inv; S.N = s->N; S.out = s->strain; S.ok = s->strain_ok;
        k_strain3<<<grid_for(s->N), kBlock, 0, s->stream>>>(S);
    } else {
        StrainParams<double2> S;
        S.pos = s->pos[s->cur]; S.ref = s->ref2; S.hdr = s->hdr; S.nbr = s->nbr; S.inv = s->d_inv; S.N = s->N; S.out = s->strain; S.ok = s->strain_ok;
        k_strain2<<<grid_for(s->N), kBlock, 0, s->stream>>>(S);
    }
    s->kernels_launched += 1;
    CUDA_TRY(s, cudaGetLastError());
    CUDA_TRY(s, cudaMemcpyAsync(E, s->strain, sizeof(double) * C * s->N, cudaMemcpyDeviceToHost, s->stream));
    if (ok) CUDA_TRY(s, cudaMemcpyAsync(ok, s->strain_ok, (size_t)s->N, cudaMemcpyDeviceToHost, s->stream));
    return check_flags(s);
}

lsm_status lsm_read_broken(lsm_sim *s, uint8_t *broken, int64_t *break_step, int64_t *n_broken) {
    CHECK_SIM(s);
    if (broken && s->M > 0) {
        k_broken_from_steps<<<grid_for(s->M), kBlock, 0, s->stream>>>(s->break_step, s->d_broken, s->M);
        s->kernels_launched += 1;
        CUDA_TRY(s, cudaMemcpyAsync(broken, s->d_broken, (size_t)s->M, cudaMemcpyDeviceToHost, s->stream));
    }
    if (break_step && s->M > 0) CUDA_TRY(s, cudaMemcpyAsync(break_step, s->break_step, sizeof(long long) * s->M, cudaMemcpyDeviceToHost, s->stream));
    std::vector<unsigned long long> nb(s->B);
    CUDA_TRY(s, cudaMemcpyAsync(nb.data(), s->nbroken, sizeof(unsigned long long) * s->B, cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    if (n_broken) { long long t = 0; for (auto q : nb) t += (long long)q; *n_broken = t; }
    return LSM_OK;
}

lsm_status lsm_read_energy(lsm_sim *s, double *U, double *KE) {
    CHECK_SIM(s);
    launch_reduce(s, s->step, -1);  // sU / sKE / f of the completed state were written by the END / INIT kernel
    CUDA_TRY(s, cudaGetLastError());
    if (U) CUDA_TRY(s, cudaMemcpyAsync(U, s->cur_U, sizeof(double) * s->B, cudaMemcpyDeviceToHost, s->stream));
    if (KE) CUDA_TRY(s, cudaMemcpyAsync(KE, s->cur_KE, sizeof(double) * s->B, cudaMemcpyDeviceToHost, s->stream));
    return check_flags(s);
}

lsm_status lsm_read_stress(lsm_sim *s, int64_t capacity, int64_t *n_samples, int64_t *step, double *R, double *U, double *KE, int64_t *nb) {
    CHECK_SIM(s);
    if (!n_samples || capacity < 0) { s->err = "n_samples is NULL or capacity < 0"; return LSM_E_INVALID; }
    const long long n = std::min<long long>(s->hist_count, capacity);   // the newest n (older unread samples are dropped)
    const long long B = s->B;
    // the last n slots of the ring, oldest first: one contiguous run, or two when the run wraps past the end of the ring
    const long long first = ((s->hist_head - n) % s->hist_cap + s->hist_cap) % s->hist_cap;
    const long long n1 = std::min<long long>(n, s->hist_cap - first), n2 = n - n1;
    auto copy_out = [&](void *dst, const void *src, size_t rec) -> cudaError_t {   // rec = bytes per sample
        if (!dst || n == 0) return cudaSuccess;
        cudaError_t e = cudaMemcpyAsync(dst, static_cast<const char *>(src) + (size_t)first * rec, (size_t)n1 * rec, cudaMemcpyDeviceToHost, s->stream);
        if (e == cudaSuccess && n2 > 0) e = cudaMemcpyAsync(static_cast<char *>(dst) + (size_t)n1 * rec, src, (size_t)n2 * rec, cudaMemcpyDeviceToHost, s->stream);
        return e;
    };
    CUDA_TRY(s, copy_out(step, s->hist_step, sizeof(long long)));
    CUDA_TRY(s, copy_out(R, s->hist_R, sizeof(double) * B * kMaxGroups * s->dim));
    CUDA_TRY(s, copy_out(U, s->hist_U, sizeof(double) * B));
    CUDA_TRY(s, copy_out(KE, s->hist_KE, sizeof(double) * B));
    CUDA_TRY(s, copy_out(nb, s->hist_nb, sizeof(long long) * B));
    *n_samples = n;
    s->hist_count = 0;
    return check_flags(s);
}

// Quasi-static driver: step in chunks that end on sample steps, look at the newest sample of the history ring (a few
// hundred bytes device -> host per chunk) and stop once every specimen's reaction has fallen below stop_fraction of its
// own running peak.  Host logic only: the steps themselves are lsm_step's.
lsm_status lsm_run_to_failure(lsm_sim *s, int64_t max_steps, int32_t group, int32_t axis, double stop_fraction, int64_t *steps_done,
                              int32_t *failed, double *peak, int64_t *peak_step) {
    CHECK_SIM(s);
    if (max_steps < 0 || group < 0 || group >= kMaxGroups || axis < 0 || axis >= s->dim || !(stop_fraction >= 0.0) || !(stop_fraction < 1.0)) { s->err = "bad arguments"; return LSM_E_INVALID; }
    if (s->sample_every <= 0) { s->err = "lsm_run_to_failure needs sample_every > 0"; return LSM_E_INVALID; }
    const long long B = s->B;
    std::vector<double> pk(B, 0.0), R((size_t)B * kMaxGroups * s->dim);
    std::vector<long long> pks(B, -1);
    std::vector<char> done(B, 0);
    long long run = 0, ndone = 0;
    while (run < max_steps && ndone < B) {
        const long long to_sample = s->sample_every - (s->step % s->sample_every);
        const long long n = std::min<long long>(to_sample, max_steps - run);
        TRY(lsm_step(s, n));
        run += n;
        if (s->step % s->sample_every != 0) break;   // max_steps ended between two samples
        const long long slot = (s->hist_head - 1 + s->hist_cap) % s->hist_cap;   // the sample lsm_step just recorded
        CUDA_TRY(s, cudaMemcpyAsync(R.data(), s->hist_R + slot * B * kMaxGroups * s->dim, sizeof(double) * R.size(), cudaMemcpyDeviceToHost, s->stream));
        TRY(check_flags(s));                          // synchronises the stream
        for (long long b = 0; b < B; ++b) {
            if (done[b]) continue;
            const double r = std::fabs(R[((size_t)b * kMaxGroups + group) * s->dim + axis]);
            if (r > pk[b]) { pk[b] = r; pks[b] = s->step; }
            else if (pk[b] > 0.0 && r < stop_fraction * pk[b]) { done[b] = 1; ++ndone; }
        }
    }
    if (steps_done) *steps_done = run;
    if (failed) *failed = ndone == B;
    for (long long b = 0; b < B; ++b) { if (peak) peak[b] = pk[b]; if (peak_step) peak_step[b] = pks[b]; }
    return LSM_OK;
}

// Strain-rate control of the paper's protocol: host logic around lsm_set_boundary plus one ramp kernel.
lsm_status lsm_set_strain_rate(lsm_sim *s, int32_t g_lo, int32_t g_hi, int32_t axis, double strain_per_step, int32_t symmetric, int32_t ramp,
                               double *gauge_length) {
    CHECK_SIM(s);
    if (s->dim != 2) { s->err = "lsm_set_strain_rate: dim = 2 only"; return LSM_E_UNSUPPORTED; }
    if (g_lo < 0 || g_lo >= kMaxGroups || g_hi < 0 || g_hi >= kMaxGroups || g_lo == g_hi || axis < 0 || axis >= s->dim || !std::isfinite(strain_per_step)) { s->err = "bad arguments"; return LSM_E_INVALID; }
    Group &lo = s->groups[g_lo], &hi = s->groups[g_hi];
    if (!lo.set || !hi.set || lo.ids.empty() || hi.ids.empty()) { s->err = "lsm_set_strain_rate: both groups must have been defined with lsm_set_boundary"; return LSM_E_INVALID; }
    // gauge length = distance between the groups' mean positions along the axis, now (sums in ascending caller id).
    // Only the members' coordinates leave the device (a gather into the read-out staging buffer, then n doubles each).
    // Everything that can be refused is refused before the first lsm_set_boundary below, so the two groups are never
    // left half redefined by a bad argument; a CUDA failure after that point makes the handle sticky-failed anyway.
    if ((long long)lo.ids.size() + (long long)hi.ids.size() > 2 * s->N || !lo.d_ids || !hi.d_ids) { s->err = "lsm_set_strain_rate: group tables are inconsistent"; return LSM_E_INVALID; }
    std::vector<double> c_lo_x(lo.ids.size()), c_hi_x(hi.ids.size());
    {
        double *scr = reinterpret_cast<double *>(s->stage[0]);     // 2 N doubles
        k_gather_axis<<<grid_for((long long)lo.ids.size()), kBlock, 0, s->stream>>>(s->pos[s->cur], lo.d_ids, (long long)lo.ids.size(), axis, scr);
        k_gather_axis<<<grid_for((long long)hi.ids.size()), kBlock, 0, s->stream>>>(s->pos[s->cur], hi.d_ids, (long long)hi.ids.size(), axis, scr + lo.ids.size());
        s->kernels_launched += 2;
        CUDA_TRY(s, cudaGetLastError());
        CUDA_TRY(s, cudaMemcpyAsync(c_lo_x.data(), scr, sizeof(double) * lo.ids.size(), cudaMemcpyDeviceToHost, s->stream));
        CUDA_TRY(s, cudaMemcpyAsync(c_hi_x.data(), scr + lo.ids.size(), sizeof(double) * hi.ids.size(), cudaMemcpyDeviceToHost, s->stream));
        TRY(check_flags(s));                                        // synchronises the stream
    }
    auto mean_of = [&](const Group &g, const std::vector<double> &val) {
        std::vector<std::pair<int32_t, double>> c(g.ids.size());
        for (size_t q = 0; q < g.ids.size(); ++q) c[q] = {s->perm.empty() ? g.ids[q] : s->perm[g.ids[q]], val[q]};
        std::sort(c.begin(), c.end(), [](const std::pair<int32_t, double> &a, const std::pair<int32_t, double> &b) { return a.first < b.first; });
        double sum = 0.0;
        for (const auto &e : c) sum += e.second;
        return sum / (double)c.size();
    };
    const double m_lo = mean_of(lo, c_lo_x), m_hi = mean_of(hi, c_hi_x), H0 = m_hi - m_lo;
    if (!(H0 > 0.0) || !std::isfinite(H0)) { s->err = "lsm_set_strain_rate: group_hi must lie above group_lo along the axis"; return LSM_E_INVALID; }
    if (gauge_length) *gauge_length = H0;
    const double du = strain_per_step * H0;
    double d_lo[3] = {0.0, 0.0, 0.0}, d_hi[3] = {0.0, 0.0, 0.0};
    d_lo[axis] = symmetric ? -0.5 * du : 0.0;
    d_hi[axis] = symmetric ? 0.5 * du : du;
    auto caller_ids = [&](const Group &g) {
        std::vector<int32_t> c(g.ids.size());
        for (size_t q = 0; q < g.ids.size(); ++q) c[q] = s->perm.empty() ? g.ids[q] : s->perm[g.ids[q]];
        return c;
    };
    const std::vector<int32_t> c_lo = caller_ids(lo), c_hi = caller_ids(hi);
    TRY(lsm_set_boundary(s, g_lo, c_lo.data(), (int64_t)c_lo.size(), LSM_MOVE, d_lo));
    TRY(lsm_set_boundary(s, g_hi, c_hi.data(), (int64_t)c_hi.size(), LSM_MOVE, d_hi));
    if (ramp) {
        const double c = symmetric ? 0.5 * (m_lo + m_hi) : m_lo;
        k_velocity_ramp<<<grid_for(s->N), kBlock, 0, s->stream>>>(s->pos[s->cur], s->vel, s->grp, s->N, axis, strain_per_step, c, s->dt);
        s->kernels_launched += 1;
        CUDA_TRY(s, cudaGetLastError());
        TRY(eval_initial(s));          // the held total force f - gamma v follows the new velocities (as after lsm_write_state)
        CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    }
    return LSM_OK;
}

lsm_status lsm_get_info(lsm_sim *s, lsm_info *info) {
    if (!s || !info) return LSM_E_INVALID;
    std::memset(info, 0, sizeof(*info));
    if (s->E_stale && s->rp_totals && s->sticky == LSM_OK) {   // compaction repacked the lists on the device since the last query
        DeviceScope scope(s->device);
        uint32_t tot = 0;
        if (cudaMemcpyAsync(&tot, s->rp_totals, sizeof(uint32_t), cudaMemcpyDeviceToHost, s->stream) == cudaSuccess &&
            cudaStreamSynchronize(s->stream) == cudaSuccess) { s->E = (long long)tot * kSlice; s->E_stale = false; }
    }
    info->n_particles = s->N; info->n_springs = s->M; info->n_half_edges_stored = s->E;
    static const int pbytes_scatter[5] = {0, 1, 8, 9, 24}, pbytes_gather[5] = {0, 1, 1, 2, 17};
    info->bytes_per_half_edge = s->force_mode == LSM_FORCE_GATHER ? (s->nbr16 && s->gather_variant == 2 ? 2 : 4) + pbytes_gather[s->pm] : 8 + pbytes_scatter[s->pm];
    info->gather_variant = s->force_mode == LSM_FORCE_GATHER ? s->gather_variant : 0;
    info->pipeline_stages = s->gather_variant == 2 ? s->L.stages : 0;
    info->step_fusion = s->res_on ? 2 : s->multi_on;
    info->cluster_size = s->res_on ? s->res_cluster : 0;
    info->window_particles = s->win_on ? s->win_cap : 0;
    info->window_stages = s->win_on ? s->LW.stages : 0;
    info->resident_smem_bytes = s->res_on ? s->RL.bytes : 0;
    info->stage_bytes = s->gather_variant == 2 ? s->L.bytes : 0;
    info->param_mode = s->pm; info->n_types = s->ntypes; info->force_mode = s->force_mode == LSM_FORCE_SCATTER ? (s->scatter_variant == 1 ? LSM_FORCE_SCATTER_WARP : s->scatter_variant == 2 ? LSM_FORCE_SCATTER_TILE : LSM_FORCE_SCATTER) : s->force_mode; info->exact = s->exact;
    info->reorder = s->reorder; info->n_batch = s->B; info->device_bytes = s->device_bytes;
    info->kernels_launched = s->kernels_launched; info->current_step = s->step;
    return LSM_OK;
}

lsm_status lsm_device_state(lsm_sim *s, const double **pos_xy, const double **vel_xy) {
    CHECK_SIM(s);
    if (pos_xy) *pos_xy = s->dim == 3 ? reinterpret_cast<const double *>(s->pos3[s->cur]) : reinterpret_cast<const double *>(s->pos[s->cur]);
    if (vel_xy) *vel_xy = s->dim == 3 ? reinterpret_cast<const double *>(s->vel3) : reinterpret_cast<const double *>(s->vel);
    return LSM_OK;
}

}  // extern "C"
