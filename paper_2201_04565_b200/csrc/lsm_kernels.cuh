// lsm_kernels.cuh -- hand-written sm_100a kernels of the lattice-spring step (see include/lsm.h).
//
// Data layout in HBM:
//   pos[2][N], vel[N], f[N], fd[N]   double2 (x,y packed: one 16-byte access per particle; streaming accesses are
//                                    fully coalesced, neighbour gathers touch one sector instead of two)
//   grp[N]                           uint8 boundary group of the particle, 0xFF = free.  For a kinematic particle the
//                                    vel slot holds its ORIGIN x0 (its velocity is du_g/dt by definition).
//   gather layout (particle-centric, sliced ELL, slice = one warp = 32 consecutive particles, tile = 8 slices = 256
//   particles = one CTA's unit of work):
//     hdr[T] (64 B per tile: slot offset of each of its 8 slices + end, live width of each slice),
//     nbr[E] int32 neighbour id; a padding slot or a dead spring holds the particle's OWN id (a spring never joins a
//     particle to itself): its gather is legal, gives r = 0 and therefore contributes nothing, with no validity test,
//     sid[E] caller spring id (cold: read only when a spring breaks or comes within the filter margin of rc),
//     per-slot parameters by ParamMode: typ[E] uint8, thr[E] uint8 = 8-bit code of (high word of rc*rc) - 1 (a
//     conservative integer filter on r^2; anything above it is decided by the exact fp64 rcS[sid]: the decision is the
//     fp64 one), kF/r0F[E].  nbr16[E] int16: the neighbour list again as offsets (neighbour - self), streamed instead
//     of nbr when every offset fits in 16 bits.
//     Slot s of lane l of slice S is entry (off[S] + s)*32 + l  -> every slot load is one coalesced 128-byte line, and
//     the slots of one tile are one contiguous range per array -> one bulk async copy per array per tile.
//     Rows are ordered by ascending caller spring id, so a particle sums its springs in the oracle's order.
//   scatter layout (the paper's spring list, re-done in SoA): si[M'], sj[M'] (si bitwise-NOT
//     once dead), per-spring parameters by ParamMode, force accumulated with fp64 RED atomics into f.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>
#include <utility>

namespace lsmk {

constexpr int kBlock = 256;
constexpr int kSlice = 32;
constexpr int kTile = 256;            // particles per tile (= kBlock): 8 slices
constexpr int kTileSlices = kTile / kSlice;
constexpr int kMaxStages = 8;
constexpr int kStreamMinB = 3;         // resident CTAs per SM the streamed kernels are compiled for (register budget)
constexpr int kRowCH = 6;              // springs of a row evaluated together (instruction-level parallelism vs registers)
typedef uint8_t thr_t;                 // per-half-edge code of the breakage filter (round 1: 16 bits; the filter only has to be
constexpr int kThrB = 1;               // conservative, so 8 bits stream half the bytes and send a few more rows to the exact pass)
constexpr int kRowCH3 = 3;             // D = 3 (32-byte positions): three at a time keep the register budget of 3 CTAs per SM
constexpr int kStreamHdrBytes = 256;   // mbarriers at the front of the streamed kernel's dynamic shared memory
constexpr uint8_t kFree = 0xFF;
constexpr int kMaxGroups = 8;
constexpr int kChunk = 2048;  // particles per reduction chunk
constexpr int kMaxTypes = 256;
constexpr int kTabStride = 6;   // gather type table, doubles per type: k, k*r0, filter word (low 32 bits), r0, rc, pad

enum ParamMode { PM_UNIFORM = 0, PM_TYPED = 1, PM_RCF = 2, PM_KRT_RCF = 3, PM_FULL = 4 };

struct __align__(16) TileHdr {          // 64 bytes per tile of 256 particles
    uint32_t off[kTileSlices + 1];     // slot offset (units of 32 entries) of each slice, and the end of the tile
    uint8_t w[kTileSlices];            // live width of each slice (shrinks under compaction)
    uint8_t pad[20];                   // pad[0..1]: window index of the tile's first particle (lsm_window.cuh)
};
static_assert(sizeof(TileHdr) == 64, "TileHdr must be 64 bytes");

struct GroupTab {
    double dux[kMaxGroups], duy[kMaxGroups], duz[kMaxGroups];   // duz: D = 3 only
    long long n0[kMaxGroups];
};

struct SpringParams {  // parameter encoding shared by the gather (per half-edge) and scatter (per spring) layouts
    const uint8_t *typ;
    const double *kF, *r0F, *rcF;      // rcF: scatter layout only
    const thr_t *thr;                  // gather layout: breakage filter per half-edge, 8 bits: the filter word
                                       // (high word of rc*rc) - 1 is thr_base + thr[e] * thr_mul, rounded down
    uint32_t thr_base, thr_mul;       // thr_mul = 1 << shift (decode = one multiply-add)
    const double *rcS;                 // gather layout: exact rc per spring, caller numbering
    const double *tab;  // scatter: [ntypes][3] = k, r0, rc;  gather: [ntypes][kTabStride] (see kTabStride)
    int ntypes;
    double k_u, r0_u, rc_u, kr0_u;
    uint32_t thr_u;
};

struct StepVar {        // what changes from one time step to the next inside a multi-step launch
    const double2 *pos_cur;
    double2 *pos_next;
    long long step;     // step number of THIS force evaluation (stamped on springs that break in it)
    uint32_t pos_s;     // GM_SMEM only: shared-memory address of (hypothetical) particle 0 in the current position buffer
};

// Where a neighbour's position is gathered from.
enum GatherMode { GM_GLOBAL_NC = 0,   // global memory through the read-only path (positions are constant during the launch)
                  GM_GLOBAL_CG = 1,   // global memory, L2 only: positions written by other CTAs earlier in the same launch
                  GM_SMEM = 2 };      // the CTA's shared-memory window (lsm_resident.cuh): own particles + ghosts

__device__ __forceinline__ double2 lds_d2(uint32_t addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

struct StepParams {
    const double2 *pos_cur;
    double2 *pos_next;
    double2 *vel, *f, *fd;
    const uint8_t *grp;
    const double *mass;
    double mass_u, inv_mass_u;
    double dt, hdt, gamma;
    long long N;
    long long step;  // step number of THIS force evaluation (stamped on springs that break in it)
    // gather layout
    const TileHdr *hdr;
    long long T;  // tiles
    int32_t *nbr;
    int16_t *nbr16;   // same list as 16-bit offsets (neighbour - self), present when every offset fits: the streamed copy
    uint16_t *widx;   // same list as window indices (lsm_window.cuh), or NULL; kept consistent by whoever kills a spring
    const int32_t *sid;
    SpringParams sp;
    // breakage bookkeeping
    long long *break_step;
    unsigned long long *nbroken;
    const long long *poff;
    int B;
    // per-particle energy scratch (written by SAMPLE variants)
    double *sU, *sKE;
    GroupTab g;
};

// ---- arithmetic: EXACT = IEEE sqrt / divide and never-contracted multiply-add (mirrors gcc -ffp-contract=off) ----
template <bool E> __device__ __forceinline__ double mul(double a, double b) { return E ? __dmul_rn(a, b) : a * b; }
template <bool E> __device__ __forceinline__ double add(double a, double b) { return E ? __dadd_rn(a, b) : a + b; }
template <bool E> __device__ __forceinline__ double sub(double a, double b) { return E ? __dsub_rn(a, b) : a - b; }
template <bool E> __device__ __forceinline__ double mad(double a, double b, double c) {  // a*b + c
    return E ? __dadd_rn(__dmul_rn(a, b), c) : fma(a, b, c);
}

// Fast-mode 1/sqrt(x) for normal x > 0: hardware seed (MUFU.RSQ64H, ~2^-20 relative) + one cubically convergent
// correction y = y0 + y0*e*(1/2 + 3/8 e), e = 1 - x*y0^2  ->  ~2^-60 before rounding, 5 fp64 ops, no special-case
// branch (the library rsqrt() carries a slow-path call per use that breaks the interleaving of a row's springs).
// x = 0 gives inf / NaN: the callers select those lanes away.
__device__ __forceinline__ double rsqrt_fast(double x) {
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x));
    const double t = x * y0;
    const double e = fma(-t, y0, 1.0);
    const double q = fma(0.375, e, 0.5);
    return fma(y0 * e, q, y0);
}

__device__ __forceinline__ int spec_of(const long long *poff, int B, long long p) {
    int lo = 0, hi = B;  // poff[lo] <= p < poff[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (poff[mid] <= p) lo = mid; else hi = mid;
    }
    return lo;
}

template <int PM> __device__ __forceinline__ void load_params(const SpringParams &sp, const double *s_tab, size_t e,
                                                              double &k, double &r0, double &rc) {
    if (PM == PM_UNIFORM) { k = sp.k_u; r0 = sp.r0_u; rc = sp.rc_u; }
    else if (PM == PM_TYPED) { int t = sp.typ[e]; k = s_tab[3 * t]; r0 = s_tab[3 * t + 1]; rc = s_tab[3 * t + 2]; }
    else if (PM == PM_RCF) { k = sp.k_u; r0 = sp.r0_u; rc = __ldg(sp.rcF + e); }
    else if (PM == PM_KRT_RCF) { int t = sp.typ[e]; k = s_tab[3 * t]; r0 = s_tab[3 * t + 1]; rc = __ldg(sp.rcF + e); }
    else { k = __ldg(sp.kF + e); r0 = __ldg(sp.r0F + e); rc = __ldg(sp.rcF + e); }
}

// One spring seen from one endpoint: d = x_other - x_self.  Returns false when the spring just broke.
// Eq. 2 with the listing's breakage test (L98).  Both endpoints compute bit-identical r
// ((-dx)^2 == dx^2), so they take the same decision without communicating.
template <bool EXACT> __device__ __forceinline__ bool spring_eval(double dx, double dy, double k, double r0, double rc,
                                                                  double &gk, double &ext) {
    const double r2 = EXACT ? add<true>(mul<true>(dx, dx), mul<true>(dy, dy)) : fma(dy, dy, dx * dx);
    double r, rinv;
    if (EXACT) { r = __dsqrt_rn(r2); rinv = 0.0; }
    else { rinv = rsqrt(r2); r = r2 * rinv; if (!(r2 > 0.0)) r = 0.0; }
    if (r > rc) return false;                       // strict '>' (Q1)
    ext = sub<EXACT>(r, r0);
    if (r == 0.0) { gk = 0.0; ext = 0.0; return true; }   // coincident endpoints: no direction, no force (Q4)
    gk = EXACT ? __ddiv_rn(mul<true>(k, ext), r) : (k * ext) * rinv;
    return true;
}

// Velocity-Verlet particle update (Eq. 3-5, half-step-velocity form L76), given the spring force
// (fx,fy) at the current positions.  KICK2: second half kick completing the step; ADVANCE: first half kick + drift of
// the next step fused behind it (the half-step velocity is what is stored between kernels); !ADVANCE: the completed
// state (v, fd).  SAMPLE: the kinetic-energy term.  particle_math is the arithmetic (the one place it is written);
// particle_update adds the stores of the direct / streamed kernels, lsm_resident.cuh its own.
struct Upd {
    double2 xn;      // ADVANCE: position after the next drift
    double2 w;       // ADVANCE: half-step velocity carried to the next force evaluation (free particles)
    double2 v;       // completed velocity of this step (free particles)
    double2 fd;      // total force f - gamma v held at force time (Q7)
    double ke;       // SAMPLE: 1/2 m |v|^2 (0 for kinematic particles, Q6)
};

template <bool EXACT, bool KICK2, bool ADVANCE, bool SAMPLE>
__device__ __forceinline__ Upd particle_math(const StepParams &P, long long step, long long p, double2 xp, double2 vh, uint8_t g, double fx, double fy) {
    Upd o;
    o.ke = 0.0;
    if (g == kFree) {
        const double fdx = sub<EXACT>(fx, mul<EXACT>(P.gamma, vh.x));  // damping with the held velocity (Q7)
        const double fdy = sub<EXACT>(fy, mul<EXACT>(P.gamma, vh.y));
        double ax, ay, m;
        if (P.mass) { m = __ldg(P.mass + p); ax = EXACT ? __ddiv_rn(fdx, m) : fdx / m; ay = EXACT ? __ddiv_rn(fdy, m) : fdy / m; }
        else { m = P.mass_u; ax = EXACT ? __ddiv_rn(fdx, m) : fdx * P.inv_mass_u; ay = EXACT ? __ddiv_rn(fdy, m) : fdy * P.inv_mass_u; }
        double2 v = vh;
        if (KICK2) { v.x = mad<EXACT>(P.hdt, ax, vh.x); v.y = mad<EXACT>(P.hdt, ay, vh.y); }  // Eq. 5, second half
        if (SAMPLE) {
            const double v2 = add<EXACT>(mul<EXACT>(v.x, v.x), mul<EXACT>(v.y, v.y));
            o.ke = mul<EXACT>(mul<EXACT>(0.5, m), v2);
        }
        o.v = v;
        o.fd = make_double2(fdx, fdy);
        if (ADVANCE) {
            if (!EXACT && KICK2 && !SAMPLE) {   // fast mode: the two half kicks of consecutive steps in one FMA (2 hdt = dt)
                o.w.x = fma(P.dt, ax, vh.x); o.w.y = fma(P.dt, ay, vh.y);
            } else {
                o.w.x = mad<EXACT>(P.hdt, ax, v.x); o.w.y = mad<EXACT>(P.hdt, ay, v.y);      // Eq. 5, first half
            }
            o.xn.x = mad<EXACT>(P.dt, o.w.x, xp.x); o.xn.y = mad<EXACT>(P.dt, o.w.y, xp.y);  // Eq. 3
        }
    } else {  // kinematic particle: vh holds its origin x0 ("boundary displacements are first applied")
        o.w = vh; o.v = vh;
        if (ADVANCE) {
            const double ns = (double)(step + 1 - P.g.n0[g]);
            o.xn = make_double2(mad<EXACT>(ns, P.g.dux[g], vh.x), mad<EXACT>(ns, P.g.duy[g], vh.y));
        } else {   // completed state: the held total force of a kinematic particle is f - gamma * (du/dt), its stored
            // velocity being du/dt (Q6, Q7); it matters only if the particle is released later (lsm_set_boundary)
            const double vkx = __ddiv_rn(P.g.dux[g], P.dt), vky = __ddiv_rn(P.g.duy[g], P.dt);
            o.fd = make_double2(sub<EXACT>(fx, mul<EXACT>(P.gamma, vkx)), sub<EXACT>(fy, mul<EXACT>(P.gamma, vky)));
        }
    }
    return o;
}

template <bool EXACT, bool KICK2, bool ADVANCE, bool SAMPLE>
__device__ __forceinline__ void particle_update(const StepParams &P, const StepVar &V, long long p, double2 xp, double2 vh, uint8_t g,
                                                double fx, double fy, double u, double2 *own_pos = nullptr, double2 *own_vel = nullptr) {
    const Upd o = particle_math<EXACT, KICK2, ADVANCE, SAMPLE>(P, V.step, p, xp, vh, g, fx, fy);
    if (SAMPLE) { P.sU[p] = u; P.sKE[p] = o.ke; }
    if (SAMPLE || !ADVANCE) P.f[p] = make_double2(fx, fy);
    if (ADVANCE) {
        V.pos_next[p] = o.xn;
        if (own_pos) *own_pos = o.xn;                    // resident tiles: the staged copy is the next step's input
        if (g == kFree) { P.vel[p] = o.w; if (own_vel) *own_vel = o.w; }
    } else {
        if (g == kFree) P.vel[p] = o.v;
        P.fd[p] = o.fd;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Fused gather step: one thread per particle.  Gathers the positions of its (<= slice width) neighbours, evaluates
// every incident spring (each spring is evaluated from both of its endpoints: twice the arithmetic, no atomics, no
// force array round trip, deterministic), applies the breakage test, then integrates.  Reads x (double-buffered),
// v, ids, parameters; writes x_next, v.  HBM bytes per step: 64 N + (2 or 4 id bytes + parameter bytes) * 2M.
// Two kernels share the row evaluation below: k_gather_step reads the slot streams straight from global memory;
// k_gather_stream (the product path) stages them tile by tile through shared memory with bulk async copies.
// ---------------------------------------------------------------------------------------------------------------
// ---- shared-memory row access with 32-bit addresses and immediate offsets (no generic-pointer arithmetic in the hot loop) ----
template <int OFF> __device__ __forceinline__ int lds_s16o(uint32_t a) { int v; asm volatile("ld.shared.s16 %0, [%1+%2];" : "=r"(v) : "r"(a), "n"(OFF)); return v; }
template <int OFF> __device__ __forceinline__ uint32_t lds_u16o(uint32_t a) { uint32_t v; asm volatile("ld.shared.u16 %0, [%1+%2];" : "=r"(v) : "r"(a), "n"(OFF)); return v; }
template <int OFF> __device__ __forceinline__ uint32_t lds_u8o(uint32_t a) { uint32_t v; asm volatile("ld.shared.u8 %0, [%1+%2];" : "=r"(v) : "r"(a), "n"(OFF)); return v; }
template <int OFF> __device__ __forceinline__ uint32_t lds_u32o(uint32_t a) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(v) : "r"(a), "n"(OFF)); return v; }
template <int OFF> __device__ __forceinline__ double lds_f64o(uint32_t a) { double v; asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(v) : "r"(a), "n"(OFF)); return v; }

// compile-time loop 0 .. N-1 (the index is usable as a template argument: immediate offsets of the loads below)
template <int N, int I = 0, class F> __device__ __forceinline__ void static_for(F &&f) {
    if constexpr (I < N) { f(std::integral_constant<int, I>{}); static_for<N, I + 1>(f); }
}

struct RowS { uint32_t nbr, thr, typ, kF, r0F; };   // shared addresses of this lane's entry in the current slot of each row array

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

__device__ __forceinline__ int lds_s32_at(uint32_t a) { int v; asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
template <int OFF> __device__ __forceinline__ int lds_s32o(uint32_t a) { int v; asm volatile("ld.shared.s32 %0, [%1+%2];" : "=r"(v) : "r"(a), "n"(OFF)); return v; }

struct RowSrc {            // where one particle's row lives: pointers already offset to (slice offset)*32 + lane
    const int32_t *nbr;    // slot s at nbr[s*32]  (global memory, or the staged shared-memory copy)
    const int16_t *nbr16;  // I16: the staged copy holds 16-bit offsets (neighbour - self) instead
    const thr_t *thr;
    const uint8_t *typ;
    const double *kF, *r0F;
    size_t e0;                // global entry index of slot 0 of this lane (for the cold paths)
};

// Row evaluation in two passes.  The FAST pass is branch-free: padding slots, dead springs and coincident endpoints
// contribute an exact 0 through selects, every slot is accumulated at once in slot order (ascending caller spring
// id; adding +-0.0 for skipped slots leaves each partial sum bit-identical), and nothing is kept per slot, so the
// springs of a chunk interleave in the fp64 pipe with few registers.  It only notes whether any spring came close to
// its breaking length.  If one did (rare), the CAREFUL pass redoes the whole row from zero, slot by slot in the
// same order with the same arithmetic, deciding each near-rc spring exactly and marking the broken ones (Q2, Q3:
// zero force already in the step they break).
//
// Breakage filter: thr = (high 32 bits of rc*rc) - 1.  For positive doubles the high word orders like the value, so
// hi32(r2) < thr proves r2 < rc^2 (1 - 2^-20): alive, with one integer compare and no conversion.  Otherwise (r within
// ~5e-7 of rc, relatively) the careful pass decides exactly as the oracle does: r = IEEE sqrt(r2) > rc in fp64.
// A per-spring rc streams the word in 16 bits: thr_base + (t << thr_shift) rounded down (the shift is chosen at create
// from the spread of rc: 2-5 bits for rc within one binade, i.e. a filter still 1e-5 fine) -- coarser, never wrong.
template <int PM> __device__ __forceinline__ void slot_params(const StepParams &P, const RowSrc &R, const double *s_tab, unsigned so,
                                                              double &k, double &r0, double &kr0, uint32_t &thr) {
    if (PM == PM_UNIFORM) { k = P.sp.k_u; r0 = P.sp.r0_u; kr0 = P.sp.kr0_u; thr = P.sp.thr_u; }
    else if (PM == PM_TYPED) {
        const int t = R.typ[so];
        const double2 kk = *reinterpret_cast<const double2 *>(s_tab + kTabStride * t);   // one 16-byte load: k, k*r0
        k = kk.x; kr0 = kk.y; r0 = s_tab[kTabStride * t + 3];
        thr = reinterpret_cast<const uint32_t *>(s_tab)[2 * (kTabStride * t + 2)];
    }
    else if (PM == PM_RCF) { k = P.sp.k_u; r0 = P.sp.r0_u; kr0 = P.sp.kr0_u; thr = P.sp.thr_base + (uint32_t)R.thr[so] * P.sp.thr_mul; }
    else if (PM == PM_KRT_RCF) {
        const int t = R.typ[so];
        const double2 kk = *reinterpret_cast<const double2 *>(s_tab + kTabStride * t);
        k = kk.x; kr0 = kk.y; r0 = s_tab[kTabStride * t + 3]; thr = P.sp.thr_base + (uint32_t)R.thr[so] * P.sp.thr_mul;
    }
    else { k = R.kF[so]; r0 = R.r0F[so]; kr0 = k * r0; thr = P.sp.thr_base + (uint32_t)R.thr[so] * P.sp.thr_mul; }
}

// Position of neighbour j.  Always a global load (every position was just streamed in by some CTA, so these are
// L1 / L2 hits); reading in-tile neighbours from the staged copy instead was measured equal on config 3 and 17 %
// slower on full lattices (a per-slot branch).  COHERENT (multi-step launches): positions written by other CTAs
// earlier in the same launch must not come from a stale L1 line -> ld.global.cg (L2 only).
template <int GM> __device__ __forceinline__ double2 gather_pos(const StepVar &V, int j) {
    if (GM == GM_SMEM) return lds_d2(V.pos_s + (uint32_t)j * 16u);
    return GM == GM_GLOBAL_CG ? __ldcg(V.pos_cur + j) : __ldg(V.pos_cur + j);
}

// One spring seen from one endpoint (Eq. 2): d = x_other - x_self, g = k (r - r0) / r.
// live: the slot holds a spring with a direction (r2 > 0: padding / dead slots gather the own position and coincident
// endpoints give no force, Q4);
// near: r2 reaches the breakage filter (see above).  Both endpoints compute bit-identical r2 ((-dx)^2 == dx^2).
template <bool EXACT, bool SAMPLE>
__device__ __forceinline__ void slot_eval(double2 xq, double2 xp, bool lower, double k, double r0, double kr0, uint32_t thr,
                                          double &dx, double &dy, double &r2, double &g, double &ue, bool &near) {
    dx = sub<EXACT>(xq.x, xp.x); dy = sub<EXACT>(xq.y, xp.y);
    // fast: the 1e-300 rides in the first FMA.  r2 is unchanged by it for every r2 above 1e-284; at r2 = 0 (padding /
    // dead slot or coincident endpoints) it makes 1/r a finite 1e150, so g is finite and g * dx = g * 0 = 0: no select.
    r2 = EXACT ? add<true>(mul<true>(dx, dx), mul<true>(dy, dy)) : fma(dy, dy, fma(dx, dx, 1e-300));
    const uint32_t hi = (uint32_t)__double2hiint(r2);
    bool live;
    ue = 0.0;
    if (EXACT) {
        const double r = __dsqrt_rn(r2);
        const double ext = sub<true>(r, r0);
        g = __ddiv_rn(mul<true>(k, ext), r);
        if (SAMPLE) ue = mul<true>(mul<true>(mul<true>(0.5, k), ext), ext);
        live = r2 > 0.0;
    } else {
        const double rinv = rsqrt_fast(r2);
        g = fma(-kr0, rinv, k);              // k (r - r0) / r = k - k r0 / r
        if (SAMPLE) { const double ext = fma(r2, rinv, -r0); ue = (0.5 * k) * ext * ext; }
        live = r2 > 1e-290;                  // false for r2 = 0 + 1e-300 (coincident / padding); used by SAMPLE only
    }
    if (EXACT) g = live ? g : 0.0;
    if (SAMPLE) ue = (live && lower) ? ue : 0.0;  // energy counted once, by the lower endpoint (Eq. 1)
    near = EXACT ? (live && hi >= thr) : (hi >= thr);   // fast: thr is far above the high word of a zero r2
}

template <int PM, bool EXACT, bool SAMPLE, int GM, bool I16, int CH>
__device__ __forceinline__ bool row_chunk(const StepParams &P, const StepVar &V, const RowSrc &R, const double *s_tab, int p, unsigned s0,
                                          double2 xp, double &fx, double &fy, double &u) {
    int nb[CH];
    double2 xq[CH];
    bool any_near = false;
    const double2 *own = V.pos_cur + p;
    asm("" : "+l"(own));   // keep the own address in a register pair: each gather address is then one wide multiply-add
#pragma unroll
    for (int c = 0; c < CH; ++c) nb[c] = I16 ? (int)R.nbr16[(s0 + c) * kSlice] : R.nbr[(s0 + c) * kSlice];   // I16: offset
#pragma unroll
    for (int c = 0; c < CH; ++c) {   // I16: address = own address + offset (one wide multiply-add per gather)
        if (I16 && GM == GM_SMEM) xq[c] = lds_d2(V.pos_s + (uint32_t)(p + nb[c]) * 16u);
        else xq[c] = I16 ? (GM == GM_GLOBAL_CG ? __ldcg(own + nb[c]) : __ldg(own + nb[c])) : gather_pos<GM>(V, nb[c]);
        if (I16) nb[c] += p;
    }
#pragma unroll
    for (int c = 0; c < CH; ++c) {
        double k, r0, kr0, dx, dy, r2, g, ue;
        uint32_t thr;
        bool near;
        slot_params<PM>(P, R, s_tab, (s0 + c) * kSlice, k, r0, kr0, thr);
        slot_eval<EXACT, SAMPLE>(xq[c], xp, p < nb[c], k, r0, kr0, thr, dx, dy, r2, g, ue, near);
        fx = mad<EXACT>(g, dx, fx);
        fy = mad<EXACT>(g, dy, fy);
        if (SAMPLE) u = add<EXACT>(u, ue);
        any_near |= near;
    }
    return any_near;
}

template <int PM, bool EXACT, bool SAMPLE, int GM, bool I16>
__device__ __forceinline__ void row_careful(const StepParams &P, const StepVar &V, const RowSrc &R, const double *s_tab, int p, unsigned w,
                                         double2 xp, double &fx, double &fy, double &u) {
    fx = 0.0; fy = 0.0; u = 0.0;
#pragma unroll 1
    for (unsigned s = 0; s < w; ++s) {
        const unsigned so = s * kSlice;
        const int nb = I16 ? p + (int)R.nbr16[so] : R.nbr[so];
        const double2 xq = gather_pos<GM>(V, nb);
        double k, r0, kr0, dx, dy, r2, g, ue;
        uint32_t thr;
        bool near;
        slot_params<PM>(P, R, s_tab, so, k, r0, kr0, thr);
        slot_eval<EXACT, SAMPLE>(xq, xp, p < nb, k, r0, kr0, thr, dx, dy, r2, g, ue, near);
        if (near) {
            const size_t e = R.e0 + so;
            double rc;
            if (PM == PM_UNIFORM) rc = P.sp.rc_u;
            else if (PM == PM_TYPED) rc = s_tab[kTabStride * R.typ[so] + 4];
            else rc = __ldg(P.sp.rcS + __ldg(P.sid + e));
            if (__dsqrt_rn(r2) > rc) {   // strict '>' (Q1)
                P.nbr[e] = p;                             // dead from now on: the slot points at its own particle
                if (P.nbr16) P.nbr16[e] = 0;
                if (P.widx) { uint16_t ob; memcpy(&ob, P.hdr[p >> 8].pad, 2); P.widx[e] = (uint16_t)(ob + (p & (kTile - 1))); }
                if (I16) const_cast<int16_t *>(R.nbr16)[so] = 0;   // and the staged copy (resident tiles are not reloaded)
                else const_cast<int32_t *>(R.nbr)[so] = p;
                if (p < nb) {
                    P.break_step[P.sid[e]] = V.step;
                    atomicAdd(P.nbroken + spec_of(P.poff, P.B, p), 1ULL);
                }
                continue;
            }
        }
        fx = mad<EXACT>(g, dx, fx);
        fy = mad<EXACT>(g, dy, fy);
        if (SAMPLE) u = add<EXACT>(u, ue);
    }
}

template <int PM, bool EXACT, bool SAMPLE, int GM, bool I16>
__device__ __forceinline__ void row_forces(const StepParams &P, const StepVar &V, const RowSrc &R, const double *s_tab, int p, unsigned w,
                                           double2 xp, double &fx, double &fy, double &u) {
    constexpr int CH = kRowCH;
    unsigned s0 = 0;
    bool any_near = false;
    for (; s0 + CH <= w; s0 += CH) any_near |= row_chunk<PM, EXACT, SAMPLE, GM, I16, CH>(P, V, R, s_tab, p, s0, xp, fx, fy, u);
    for (; s0 < w; ++s0) any_near |= row_chunk<PM, EXACT, SAMPLE, GM, I16, 1>(P, V, R, s_tab, p, s0, xp, fx, fy, u);
    if (any_near) row_careful<PM, EXACT, SAMPLE, GM, I16>(P, V, R, s_tab, p, w, xp, fx, fy, u);
}

// The same chunk for the streamed kernel's consumers: the row comes from the pipeline stage through 32-bit shared
// addresses with immediate offsets (no generic-pointer arithmetic per slot), the neighbour positions from global memory.
template <int PM, bool EXACT, bool SAMPLE, int GM, bool I16, int CH>
__device__ __forceinline__ bool row_chunk_g(const StepParams &P, const StepVar &V, const RowS &A, uint32_t tab_s, int p, double2 xp,
                                            double &fx, double &fy, double &u) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    constexpr bool kHasThr = (PM == PM_RCF || PM == PM_KRT_RCF || PM == PM_FULL);
    int nb[CH];
    double2 xq[CH];
    bool any_near = false;
    const double2 *own = V.pos_cur + p;
    asm("" : "+l"(own));   // keep the own address in a register pair: each gather address is then one wide multiply-add
    static_for<CH>([&](auto ic) { constexpr int C = decltype(ic)::value; nb[C] = I16 ? lds_s16o<C * kSlice * 2>(A.nbr) : lds_s32o<C * kSlice * 4>(A.nbr); });
#pragma unroll
    for (int c = 0; c < CH; ++c) {
        xq[c] = I16 ? (GM == GM_GLOBAL_CG ? __ldcg(own + nb[c]) : __ldg(own + nb[c])) : gather_pos<GM>(V, nb[c]);
        if (I16) nb[c] += p;
    }
    static_for<CH>([&](auto ic) {
        constexpr int C = decltype(ic)::value;
        double k, r0 = 0.0, kr0, dx, dy, r2, g, ue;
        uint32_t thr;
        bool near;
        if constexpr (kTab) {
            const uint32_t ta = tab_s + lds_u8o<C * kSlice>(A.typ) * (uint32_t)(kTabStride * 8);
            const double2 kk = lds_d2(ta);
            k = kk.x; kr0 = kk.y;
            if (EXACT || SAMPLE) r0 = lds_f64o<24>(ta);
            thr = PM == PM_TYPED ? lds_u32o<16>(ta) : P.sp.thr_base + lds_u8o<C * kSlice * kThrB>(A.thr) * P.sp.thr_mul;
        } else if constexpr (PM == PM_FULL) {
            k = lds_f64o<C * kSlice * 8>(A.kF); r0 = lds_f64o<C * kSlice * 8>(A.r0F); kr0 = k * r0;
            thr = P.sp.thr_base + lds_u8o<C * kSlice * kThrB>(A.thr) * P.sp.thr_mul;
        } else {
            k = P.sp.k_u; r0 = P.sp.r0_u; kr0 = P.sp.kr0_u;
            thr = kHasThr ? P.sp.thr_base + lds_u8o<C * kSlice * kThrB>(A.thr) * P.sp.thr_mul : P.sp.thr_u;
        }
        slot_eval<EXACT, SAMPLE>(xq[C], xp, p < nb[C], k, r0, kr0, thr, dx, dy, r2, g, ue, near);
        fx = mad<EXACT>(g, dx, fx);
        fy = mad<EXACT>(g, dy, fy);
        if (SAMPLE) u = add<EXACT>(u, ue);
        any_near |= near;
    });
    return any_near;
}

// Direct variant: block = tile, every stream read from global memory by the thread that needs it.
template <int PM, bool EXACT, bool KICK2, bool ADVANCE, bool SAMPLE>
__global__ void __launch_bounds__(kBlock) k_gather_step(const StepParams P) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    __shared__ __align__(16) double s_tab[kTab ? kTabStride * kMaxTypes : 1];
    if (kTab) {
        for (int i = threadIdx.x; i < kTabStride * P.sp.ntypes; i += kBlock) s_tab[i] = P.sp.tab[i];
        __syncthreads();
    }
    const long long p = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (p >= P.N) return;
    const int wi = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const TileHdr *h = P.hdr + blockIdx.x;
    const unsigned w = h->w[wi];
    const size_t e0 = (size_t)h->off[wi] * kSlice + lane;
    const double2 xp = P.pos_cur[p];
    const double2 vh = P.vel[p];
    const uint8_t g = P.grp[p];
    RowSrc R;
    R.nbr = P.nbr + e0; R.nbr16 = nullptr; R.thr = P.sp.thr + e0; R.typ = P.sp.typ + e0; R.kF = P.sp.kF + e0; R.r0F = P.sp.r0F + e0;
    R.e0 = e0;
    double fx = 0.0, fy = 0.0, u = 0.0;
    const StepVar V{P.pos_cur, P.pos_next, P.step, 0u};
    row_forces<PM, EXACT, SAMPLE, GM_GLOBAL_NC, false>(P, V, R, s_tab, (int)p, w, xp, fx, fy, u);
    particle_update<EXACT, KICK2, ADVANCE, SAMPLE>(P, V, p, xp, vh, g, fx, fy, u);
}

// ---- mbarrier / bulk-copy primitives (PTX; sm_90+ async proxy: the copy engine moves the bytes, no registers) ----
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
    const uint32_t a = smem_u32(bar);
    uint32_t ok;
    do {
        // the suspend-time hint (ns) lets the hardware park the thread until the phase completes instead of re-polling
        asm volatile("{\n\t.reg .pred q;\n\tmbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, q;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity), "r"(0x989680u) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// Grid barrier of the cooperative multi-step launches, one thread per CTA: a release-add on a global arrival counter (this
// CTA's stores, observed through its step barrier, become visible first), then acquire-polls until every CTA has arrived.
__device__ __forceinline__ void grid_arrive_and_wait(unsigned long long *ctr, unsigned long long target) {
    asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(ctr) : "memory");
    unsigned long long v;
    do { asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(ctr) : "memory"); } while (v < target);
}

struct StageLayout {      // byte offsets of the staged arrays inside one pipeline stage (all multiples of 128)
    int pos, vel, hdr, grp, nbr, thr, typ, kF, r0F;
    int bytes;            // stage size
    int stages;           // pipeline depth
    int first;            // offset of stage 0 in dynamic shared memory (after the barriers and the type table)
};

// Streamed variant (product path).  Persistent CTAs (grid = CTAs/SM x SMs) walk the tiles round-robin.  Warp 8 is the
// producer: one lane arms the stage's mbarrier with the byte count and issues one bulk async copy per array
// (own x, own v, group bytes, tile header, neighbour ids, parameters); warps 0..7 are the consumers (one thread per
// particle).  The bytes in flight per SM are (stages - 1) x stage size x CTAs/SM, independent of registers and
// occupancy; the only latency the consumers see is the neighbour-position gather (L1 / L2 hits).
//
// MULTI: the launch advances M.nsteps time steps (cooperative launch, all CTAs resident).  Between two steps every
// CTA passes a grid barrier: its consumer warps publish their stores (__threadfence) and arrive on a CTA-local
// mbarrier; the producer lane waits for it, arrives on a global counter, spins until all CTAs of this step have
// arrived, orders the generic-proxy writes before its next bulk copies (fence.proxy.async) and refills the pipeline
// from the swapped position buffers.  Small (L2-resident, launch-bound) problems step ~2x faster this way.
struct MultiParams {
    int nsteps;                       // time steps in this launch (1 when !MULTI)
    unsigned long long *gbar;         // global arrival counter (monotonic across launches)
    unsigned long long gbar_base;     // its value before this launch
    int resident;                     // 1: every CTA's tiles fit in its pipeline stages -> loaded once, kept in shared
                                      //    memory for the whole launch (rows, own x and v); later steps copy nothing
    double2 *pos_a, *pos_b;           // step i reads pos_a / writes pos_b when i is even, the reverse when odd
};

}  // namespace lsmk
#include "lsm_rows3.cuh"
namespace lsmk {

// D = 3: the same pipeline with 32-byte {x, y, z, 0} position / velocity records (the pointers of StepParams / StepVar /
// MultiParams then address double4) and the row functions of lsm_rows3.cuh.
template <int PM, bool EXACT, bool KICK2, bool ADVANCE, bool SAMPLE, bool MULTI, bool I16, int D = 2>
__global__ void __launch_bounds__(kTile + 32, kStreamMinB) k_gather_stream(const StepParams P, const StageLayout L, const MultiParams M) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    constexpr bool kHasThr = (PM == PM_RCF || PM == PM_KRT_RCF || PM == PM_FULL);
    constexpr bool kHasTyp = kTab;
    constexpr bool kHasKR = (PM == PM_FULL);
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);          // [kMaxStages]
    uint64_t *empty = full + kMaxStages;                            // [kMaxStages]
    uint64_t *stepdone = empty + kMaxStages;                        // MULTI: all consumer warps of this CTA finished the step
    uint64_t *go = stepdone + 1;                                    // MULTI resident: the grid barrier has been passed
    double *s_tab = reinterpret_cast<double *>(smem + kStreamHdrBytes);         // [kTabStride * ntypes] when kTab
    unsigned char *stage0 = smem + L.first;
    const int tid = threadIdx.x, wi = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < L.stages; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, kTileSlices); }
        if (MULTI) { mbar_init(stepdone, kTileSlices); mbar_init(go, 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (kTab) for (int i = tid; i < kTabStride * P.sp.ntypes; i += kTile + 32) s_tab[i] = P.sp.tab[i];
    __syncthreads();
    const int nsteps = MULTI ? M.nsteps : 1;
    constexpr int kVB = D == 3 ? 32 : 16;   // bytes of one position / velocity record

    if (wi == kTileSlices) {  // ---------------- producer warp ----------------
        if (lane == 0) {
            int s = 0; unsigned u = 0;
            for (int it = 0; it < nsteps; ++it) {
                const double2 *pos_cur = MULTI ? ((it & 1) ? M.pos_b : M.pos_a) : P.pos_cur;
                if (MULTI && it > 0) {  // grid barrier: every CTA has finished (and published) step it-1
                    mbar_wait(stepdone, (it - 1) & 1);
                    grid_arrive_and_wait(M.gbar, M.gbar_base + (unsigned long long)it * gridDim.x);
                    asm volatile("fence.proxy.async;" ::: "memory");
                    if (M.resident) { mbar_arrive(go); continue; }   // nothing to copy: the consumers own the staged tiles
                }
                uint32_t o0n = 0, o8n = 0;
                if ((long long)blockIdx.x < P.T) { o0n = __ldg(&P.hdr[blockIdx.x].off[0]); o8n = __ldg(&P.hdr[blockIdx.x].off[kTileSlices]); }
                for (long long t = blockIdx.x; t < P.T; t += gridDim.x) {
                    const TileHdr *h = P.hdr + t;
                    const uint32_t o0 = o0n, ns = o8n - o0n;
                    if (t + gridDim.x < P.T) { o0n = __ldg(&h[gridDim.x].off[0]); o8n = __ldg(&h[gridDim.x].off[kTileSlices]); }  // next tile's extent, ahead of the wait
                    if (u > 0) mbar_wait(empty + s, (u - 1) & 1);
                    constexpr unsigned kIdB = I16 ? 2 : 4;   // bytes per streamed neighbour id
                    unsigned bytes = 2 * kTile * kVB + kTile + 64 + ns * (kSlice * kIdB);
                    if (kHasThr) bytes += ns * (kSlice * kThrB);
                    if (kHasTyp) bytes += ns * kSlice;
                    if (kHasKR) bytes += 2 * ns * (kSlice * 8);
                    unsigned char *b = stage0 + (size_t)s * L.bytes;
                    mbar_expect_tx(full + s, bytes);
                    bulk_g2s(b + L.pos, reinterpret_cast<const char *>(pos_cur) + t * (kTile * kVB), kTile * kVB, full + s);
                    bulk_g2s(b + L.vel, reinterpret_cast<const char *>(P.vel) + t * (kTile * kVB), kTile * kVB, full + s);
                    bulk_g2s(b + L.grp, P.grp + t * kTile, kTile, full + s);
                    bulk_g2s(b + L.hdr, h, 64, full + s);
                    if (ns) {
                        const size_t e = (size_t)o0 * kSlice;
                        if (I16) bulk_g2s(b + L.nbr, P.nbr16 + e, ns * (kSlice * 2), full + s);
                        else bulk_g2s(b + L.nbr, P.nbr + e, ns * (kSlice * 4), full + s);
                        if (kHasThr) bulk_g2s(b + L.thr, P.sp.thr + e, ns * (kSlice * kThrB), full + s);
                        if (kHasTyp) bulk_g2s(b + L.typ, P.sp.typ + e, ns * kSlice, full + s);
                        if (kHasKR) {
                            bulk_g2s(b + L.kF, P.sp.kF + e, ns * (kSlice * 8), full + s);
                            bulk_g2s(b + L.r0F, P.sp.r0F + e, ns * (kSlice * 8), full + s);
                        }
                    }
                    if (++s == L.stages) { s = 0; ++u; }
                }
            }
        }
        return;
    }
    // ---------------- consumer warps: thread = particle ----------------
    int s = 0; unsigned u = 0;
    for (int it = 0; it < nsteps; ++it) {
        StepVar V;
        V.pos_cur = MULTI ? ((it & 1) ? M.pos_b : M.pos_a) : P.pos_cur;
        V.pos_next = MULTI ? ((it & 1) ? M.pos_a : M.pos_b) : P.pos_next;
        V.step = P.step + it;
        V.pos_s = 0u;
        const bool kept = MULTI && M.resident && it > 0;   // tiles already in shared memory (stage i = i-th tile of this CTA)
        if (kept) { mbar_wait(go, (it - 1) & 1); s = 0; }
        for (long long t = blockIdx.x; t < P.T; t += gridDim.x) {
            if (!kept) mbar_wait(full + s, u & 1);
            unsigned char *b = stage0 + (size_t)s * L.bytes;
            const TileHdr *h = reinterpret_cast<const TileHdr *>(b + L.hdr);
            const long long p = t * kTile + tid;
            if (p < P.N) {
                const unsigned w = h->w[wi];
                const unsigned rel = (h->off[wi] - h->off[0]) * kSlice + lane;
                RowSrc R;
                R.nbr = reinterpret_cast<const int32_t *>(b + L.nbr) + rel;
                R.nbr16 = reinterpret_cast<const int16_t *>(b + L.nbr) + rel;
                R.thr = reinterpret_cast<const thr_t *>(b + L.thr) + rel;
                R.typ = (b + L.typ) + rel;
                R.kF = reinterpret_cast<const double *>(b + L.kF) + rel;
                R.r0F = reinterpret_cast<const double *>(b + L.r0F) + rel;
                R.e0 = (size_t)h->off[wi] * kSlice + lane;
                if constexpr (D == 3) {
                    const double4 xp = reinterpret_cast<const double4 *>(b + L.pos)[tid];
                    double fx = 0.0, fy = 0.0, fz = 0.0, uu = 0.0;
                    row_forces3<PM, EXACT, SAMPLE, MULTI, I16>(P, V, R, s_tab, (int)p, w, xp, fx, fy, fz, uu);
                    const double4 vh = reinterpret_cast<const double4 *>(b + L.vel)[tid];
                    const uint8_t g = (b + L.grp)[tid];
                    if (MULTI && M.resident)
                        particle_update3<EXACT, KICK2, ADVANCE, SAMPLE>(P, V, p, xp, vh, g, fx, fy, fz, uu, reinterpret_cast<double4 *>(b + L.pos) + tid,
                                                                        reinterpret_cast<double4 *>(b + L.vel) + tid);
                    else
                        particle_update3<EXACT, KICK2, ADVANCE, SAMPLE>(P, V, p, xp, vh, g, fx, fy, fz, uu);
                } else {
                    const double2 xp = reinterpret_cast<const double2 *>(b + L.pos)[tid];
                    double fx = 0.0, fy = 0.0, uu = 0.0;
                    if constexpr (MULTI) {   // cooperative multi-step launches: measured 3.5 % faster with the generic-pointer row code
                        row_forces<PM, EXACT, SAMPLE, GM_GLOBAL_CG, I16>(P, V, R, s_tab, (int)p, w, xp, fx, fy, uu);
                    } else {   // the row: chunks of kRowCH springs through 32-bit shared addresses, then the careful pass if needed
                        constexpr int GMv = GM_GLOBAL_NC;
                        constexpr unsigned kIdB = I16 ? 2 : 4;
                        const uint32_t b_s = smem_u32(b);
                        RowS A;
                        A.nbr = b_s + (uint32_t)L.nbr + rel * kIdB; A.thr = b_s + (uint32_t)L.thr + rel * kThrB; A.typ = b_s + (uint32_t)L.typ + rel;
                        A.kF = b_s + (uint32_t)L.kF + rel * 8; A.r0F = b_s + (uint32_t)L.r0F + rel * 8;
                        const uint32_t tab_s = smem_u32(s_tab);
                        constexpr int CH = kRowCH;
                        bool any_near = false;
                        unsigned s0 = 0;
                        for (; s0 + CH <= w; s0 += CH) {
                            any_near |= row_chunk_g<PM, EXACT, SAMPLE, GMv, I16, CH>(P, V, A, tab_s, (int)p, xp, fx, fy, uu);
                            A.nbr += CH * kSlice * kIdB; A.thr += CH * kSlice * kThrB; A.typ += CH * kSlice; A.kF += CH * kSlice * 8; A.r0F += CH * kSlice * 8;
                        }
                        for (; s0 < w; ++s0) {
                            any_near |= row_chunk_g<PM, EXACT, SAMPLE, GMv, I16, 1>(P, V, A, tab_s, (int)p, xp, fx, fy, uu);
                            A.nbr += kSlice * kIdB; A.thr += kSlice * kThrB; A.typ += kSlice; A.kF += kSlice * 8; A.r0F += kSlice * 8;
                        }
                        if (any_near) row_careful<PM, EXACT, SAMPLE, GMv, I16>(P, V, R, s_tab, (int)p, w, xp, fx, fy, uu);
                    }
                    const double2 vh = reinterpret_cast<const double2 *>(b + L.vel)[tid];
                    const uint8_t g = (b + L.grp)[tid];
                    if (MULTI && M.resident)
                        particle_update<EXACT, KICK2, ADVANCE, SAMPLE>(P, V, p, xp, vh, g, fx, fy, uu, reinterpret_cast<double2 *>(b + L.pos) + tid,
                                                                       reinterpret_cast<double2 *>(b + L.vel) + tid);
                    else
                        particle_update<EXACT, KICK2, ADVANCE, SAMPLE>(P, V, p, xp, vh, g, fx, fy, uu);
                }
            }
            __syncwarp();
            if (lane == 0 && !(MULTI && M.resident)) mbar_arrive(empty + s);
            if (++s == L.stages) { s = 0; ++u; }
        }
        if (MULTI && it + 1 < nsteps) {  // tell the producer this warp is done with the step.  No fence here: the warp's
            // stores are ordered before lane 0's arrive (release.cta) by __syncwarp, the producer's wait acquires them,
            // and ITS __threadfence before the global arrival is cumulative -- the pattern of a cooperative grid sync
            // (one fencing thread per CTA).  A fence per warp cost 0.3-0.6 us per step.
            __syncwarp();
            if (lane == 0) mbar_arrive(stepdone);
        }
    }
}

// First half kick + drift from a completed state (v, fd): the first kernel of every lsm_step call.
template <bool EXACT>
__global__ void __launch_bounds__(kBlock) k_start(const StepParams P) {
    const long long p = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (p >= P.N) return;
    const double2 xp = P.pos_cur[p];
    const double2 v = P.vel[p];
    const uint8_t g = P.grp[p];
    if (g == kFree) {
        const double2 fd = P.fd[p];
        double ax, ay;
        if (P.mass) { const double m = __ldg(P.mass + p); ax = EXACT ? __ddiv_rn(fd.x, m) : fd.x / m; ay = EXACT ? __ddiv_rn(fd.y, m) : fd.y / m; }
        else { ax = EXACT ? __ddiv_rn(fd.x, P.mass_u) : fd.x * P.inv_mass_u; ay = EXACT ? __ddiv_rn(fd.y, P.mass_u) : fd.y * P.inv_mass_u; }
        double2 w, xn;
        w.x = mad<EXACT>(P.hdt, ax, v.x); w.y = mad<EXACT>(P.hdt, ay, v.y);
        xn.x = mad<EXACT>(P.dt, w.x, xp.x); xn.y = mad<EXACT>(P.dt, w.y, xp.y);
        P.pos_next[p] = xn;
        P.vel[p] = w;
    } else {
        const double ns = (double)(P.step + 1 - P.g.n0[g]);
        P.pos_next[p] = make_double2(mad<EXACT>(ns, P.g.dux[g], v.x), mad<EXACT>(ns, P.g.duy[g], v.y));
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Scatter path = the paper's design (one thread per spring, atomicAdd into f: PAPER.md:L88-L111) re-done with
// packed fp64 positions, a dead bit instead of k = 0, and RED.ADD.F64 (no return value).  Kept as the measured
// "paper design" row; the fused gather kernel above is the product path.
// ---------------------------------------------------------------------------------------------------------------
struct ScatterParams {
    int32_t *si;
    const int32_t *sj;
    const int32_t *sid;
    SpringParams sp;
    long long M;
    double *sUs;  // per-spring energy scratch (SAMPLE)
    // aggregated variants (springs stored as (lower endpoint, upper endpoint), sorted by the lower one)
    const int32_t *own_off;    // [N+1] springs whose lower endpoint is p: [own_off[p], own_off[p+1])
    const int32_t *jl_off;     // [N+1] springs whose upper endpoint is p and whose lower endpoint lies in p's tile ...
    const int32_t *jl_idx;     // ... as indices into the spring list
    const int32_t *tile_off;   // [tiles+1] spring range of each tile of kScatterTile particles
    long long N;
};
constexpr int kScatterTile = 1024;     // particles per CTA of the shared-memory tile variant
constexpr int kScatterTileThreads = 512;

template <int PM, bool SAMPLE>
__global__ void __launch_bounds__(kBlock) k_spring_scatter(const StepParams P, const ScatterParams S) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    __shared__ double s_tab[kTab ? 3 * kMaxTypes : 1];
    if (kTab) {
        for (int i = threadIdx.x; i < 3 * S.sp.ntypes; i += kBlock) s_tab[i] = S.sp.tab[i];
        __syncthreads();
    }
    const long long e = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (e >= S.M) return;
    const int i = S.si[e];
    if (i < 0) { if (SAMPLE) S.sUs[e] = 0.0; return; }
    const int j = S.sj[e];
    const double2 xi = P.pos_cur[i], xj = P.pos_cur[j];
    double k, r0, rc;
    load_params<PM>(S.sp, s_tab, (size_t)e, k, r0, rc);
    const double dx = xj.x - xi.x, dy = xj.y - xi.y;
    double gk, ext;
    if (spring_eval<false>(dx, dy, k, r0, rc, gk, ext)) {
        const double gx = gk * dx, gy = gk * dy;
        double *fi = reinterpret_cast<double *>(P.f + i), *fj = reinterpret_cast<double *>(P.f + j);
        atomicAdd(fi, gx); atomicAdd(fi + 1, gy);       // REDG.E.ADD.F64 (result unused)
        atomicAdd(fj, -gx); atomicAdd(fj + 1, -gy);
        if (SAMPLE) S.sUs[e] = 0.5 * k * ext * ext;
    } else {
        S.si[e] = ~i;
        P.break_step[S.sid[e]] = P.step;
        atomicAdd(P.nbroken + spec_of(P.poff, P.B, i), 1ULL);
        if (SAMPLE) S.sUs[e] = 0.0;
    }
}

// Scatter variant 2 (north_star: "warp-aggregated atomics"): springs are stored as (lower endpoint, upper endpoint) and
// sorted by the lower one, so the ~3 springs of a particle sit in consecutive lanes.  Lower side: segmented shuffle
// reduction over the run of equal ids, one RED pair per particle per warp.  Upper side: one RED pair per spring.  Same
// arithmetic per spring as k_spring_scatter; the order of the REDs across warps is not fixed.
template <int PM, bool SAMPLE>
__global__ void __launch_bounds__(kBlock) k_spring_scatter_warp(const StepParams P, const ScatterParams S) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    __shared__ double s_tab[kTab ? 3 * kMaxTypes : 1];
    if (kTab) {
        for (int i = threadIdx.x; i < 3 * S.sp.ntypes; i += kBlock) s_tab[i] = S.sp.tab[i];
        __syncthreads();
    }
    const long long e = (long long)blockIdx.x * kBlock + threadIdx.x;
    const unsigned lane = threadIdx.x & 31;
    int i = -1, j = -1;
    double gx = 0.0, gy = 0.0;
    if (e < S.M) {
        i = S.si[e];
        if (i < 0) { if (SAMPLE) S.sUs[e] = 0.0; i = ~i; }          // dead: stays in its particle's run, contributes 0
        else {
            j = S.sj[e];
            const double2 xi = P.pos_cur[i], xj = P.pos_cur[j];
            double k, r0, rc;
            load_params<PM>(S.sp, s_tab, (size_t)e, k, r0, rc);
            const double dx = xj.x - xi.x, dy = xj.y - xi.y;
            double gk, ext;
            if (spring_eval<false>(dx, dy, k, r0, rc, gk, ext)) {
                gx = gk * dx; gy = gk * dy;
                if (SAMPLE) S.sUs[e] = 0.5 * k * ext * ext;
            } else {
                S.si[e] = ~i;
                P.break_step[S.sid[e]] = P.step;
                atomicAdd(P.nbroken + spec_of(P.poff, P.B, i), 1ULL);
                if (SAMPLE) S.sUs[e] = 0.0;
                j = -1;
            }
        }
    }
    // lower endpoint: runs of equal i are contiguous lanes (sorted list; dead springs keep their place) -> segmented
    // reduction by shuffle-down
    const unsigned run = __match_any_sync(0xffffffffu, i);
    double ax = gx, ay = gy;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double tx = __shfl_down_sync(0xffffffffu, ax, o), ty = __shfl_down_sync(0xffffffffu, ay, o);
        if (lane + o < 32 && ((run >> (lane + o)) & 1u)) { ax += tx; ay += ty; }
    }
    if (i >= 0 && (lane == 0 || !((run >> (lane - 1)) & 1u))) {     // first lane of its run
        double *fi = reinterpret_cast<double *>(P.f + i);
        atomicAdd(fi, ax); atomicAdd(fi + 1, ay);
    }
    // upper endpoint: one RED pair per spring.  (Aggregating these too -- __match_any_sync on j, peers summed through
    // __fns / __shfl loops -- halved the RED sectors again but quadrupled the instruction count: 129 us against 115 us
    // for the plain kernel on config 3, profiles/r2_accumulation_variants.md.)
    if (j >= 0) {
        double *fj = reinterpret_cast<double *>(P.f + j);
        atomicAdd(fj, -gx); atomicAdd(fj + 1, -gy);
    }
}

// Scatter variant 3 (north_star: "shared-memory tile accumulation"): a CTA owns kScatterTile consecutive particles and
// the springs whose lower endpoint is one of them (a contiguous range of the sorted list).  Phase A, one thread per
// spring: evaluate it ONCE and park g*d in the spring's own shared-memory slot (plain STS: no shared-memory atomics,
// which are compare-and-swap loops for fp64 on sm_100a); a spring whose upper endpoint belongs to another tile spills
// its reaction with a global RED.  Phase B, one thread per particle: add the slots of the springs it is the lower
// endpoint of (a contiguous run), subtract those it is the upper endpoint of (index list), one RED pair per particle
// into f (other tiles' spills land there too).
template <int PM, bool SAMPLE>
__global__ void __launch_bounds__(kScatterTileThreads) k_spring_scatter_tile(const StepParams P, const ScatterParams S) {
    constexpr bool kTab = (PM == PM_TYPED || PM == PM_KRT_RCF);
    __shared__ double s_tab[kTab ? 3 * kMaxTypes : 1];
    extern __shared__ __align__(16) unsigned char dyn[];
    double2 *G = reinterpret_cast<double2 *>(dyn);
    if (kTab) for (int i = threadIdx.x; i < 3 * S.sp.ntypes; i += kScatterTileThreads) s_tab[i] = S.sp.tab[i];
    const long long p0 = (long long)blockIdx.x * kScatterTile, p1 = min(S.N, p0 + kScatterTile);
    const int s0 = S.tile_off[blockIdx.x], s1 = S.tile_off[blockIdx.x + 1];
    __syncthreads();
    for (int e = s0 + threadIdx.x; e < s1; e += kScatterTileThreads) {
        double2 gd = make_double2(0.0, 0.0);
        const int i = S.si[e];
        if (i < 0) { if (SAMPLE) S.sUs[e] = 0.0; }
        else {
            const int j = S.sj[e];
            const double2 xi = P.pos_cur[i], xj = P.pos_cur[j];
            double k, r0, rc;
            load_params<PM>(S.sp, s_tab, (size_t)e, k, r0, rc);
            const double dx = xj.x - xi.x, dy = xj.y - xi.y;
            double gk, ext;
            if (spring_eval<false>(dx, dy, k, r0, rc, gk, ext)) {
                gd = make_double2(gk * dx, gk * dy);
                if (SAMPLE) S.sUs[e] = 0.5 * k * ext * ext;
                if (j >= p1) {                                    // upper endpoint in another tile: spill
                    double *fj = reinterpret_cast<double *>(P.f + j);
                    atomicAdd(fj, -gd.x); atomicAdd(fj + 1, -gd.y);
                }
            } else {
                S.si[e] = ~i;
                P.break_step[S.sid[e]] = P.step;
                atomicAdd(P.nbroken + spec_of(P.poff, P.B, i), 1ULL);
                if (SAMPLE) S.sUs[e] = 0.0;
            }
        }
        G[e - s0] = gd;
    }
    __syncthreads();
    for (long long p = p0 + threadIdx.x; p < p1; p += kScatterTileThreads) {
        double fx = 0.0, fy = 0.0;
        for (int e = S.own_off[p]; e < S.own_off[p + 1]; ++e) { const double2 g = G[e - s0]; fx += g.x; fy += g.y; }
        for (int q = S.jl_off[p]; q < S.jl_off[p + 1]; ++q) { const double2 g = G[S.jl_idx[q] - s0]; fx -= g.x; fy -= g.y; }
        double *fp = reinterpret_cast<double *>(P.f + p);
        atomicAdd(fp, fx); atomicAdd(fp + 1, fy);
    }
}

// Integrate pass of the scatter path: consumes f (and zeroes it for the next spring pass when ADVANCE).
template <bool KICK2, bool ADVANCE, bool SAMPLE>
__global__ void __launch_bounds__(kBlock) k_integrate(const StepParams P) {
    const long long p = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (p >= P.N) return;
    const double2 xp = P.pos_cur[p];
    const double2 vh = P.vel[p];
    const uint8_t g = P.grp[p];
    const double2 f = P.f[p];
    // in-place variant: pos_next == pos_cur for this path
    particle_update<false, KICK2, ADVANCE, SAMPLE>(P, StepVar{P.pos_cur, P.pos_next, P.step, 0u}, p, xp, vh, g, f.x, f.y, 0.0);
    if (ADVANCE && !SAMPLE) P.f[p] = make_double2(0.0, 0.0);
}

__global__ void __launch_bounds__(kBlock) k_zero_f(double2 *f, long long N) {
    const long long p = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (p < N) f[p] = make_double2(0.0, 0.0);
}

// ---------------------------------------------------------------------------------------------------------------
// Reductions (a6): deterministic two-level sums.  Level 1: one block per chunk of <= kChunk particles of one
// specimen.  Level 2: one warp per specimen sums its chunk partials and its boundary groups' forces in a fixed order.
// ---------------------------------------------------------------------------------------------------------------
struct ReduceParams {
    const double *sU, *sKE;
    const double2 *f;
    const long long *chunk_lo, *chunk_hi;  // [nchunks]
    const int *spec_chunk_off;             // [B+1]
    double *part;                          // [nchunks][2]
    const int32_t *gids[kMaxGroups];       // members of each group, internal ids, sorted
    const long long *gseg[kMaxGroups];     // [B+1] segment of each specimen inside gids[g]
    const unsigned long long *nbroken;
    int B;
    long long step;
    // outputs
    long long *out_step;                   // scalar or NULL
    double *out_R;                         // [B][8][2] or NULL
    double *out_U, *out_KE;                // [B]
    long long *out_nb;                     // [B] or NULL
    int *flags;                            // bit 0: non-finite energy
    // scatter path: per-spring energies summed per specimen
    const double *sUs;
    const long long *soff_list;            // [B+1] specimen segments of the (sorted) spring list, or NULL
};

__global__ void __launch_bounds__(kBlock) k_reduce_chunks(const ReduceParams R) {
    __shared__ double sh[2][kBlock];
    const int c = blockIdx.x;
    const long long lo = R.chunk_lo[c], hi = R.chunk_hi[c];
    double u = 0.0, ke = 0.0;
    for (long long p = lo + threadIdx.x; p < hi; p += kBlock) { u += R.sU[p]; ke += R.sKE[p]; }
    sh[0][threadIdx.x] = u; sh[1][threadIdx.x] = ke;
    __syncthreads();
    for (int s = kBlock / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) { sh[0][threadIdx.x] += sh[0][threadIdx.x + s]; sh[1][threadIdx.x] += sh[1][threadIdx.x + s]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { R.part[2 * c] = sh[0][0]; R.part[2 * c + 1] = sh[1][0]; }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Fixed-order block sum (256 threads): shuffle tree inside each warp, then the 8 warp sums in warp order.
__device__ __forceinline__ double block_sum(double v, double *sh8) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh8[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < kBlock / 32; ++w) t += sh8[w];
    return t;
}

// One block per specimen: sums its chunk partials and its boundary groups' spring forces in a fixed order.
__global__ void __launch_bounds__(kBlock) k_finalize_sample(const ReduceParams R) {
    __shared__ double sh8[kBlock / 32];
    const int b = blockIdx.x;
    double u = 0.0, ke = 0.0;
    for (int c = R.spec_chunk_off[b] + threadIdx.x; c < R.spec_chunk_off[b + 1]; c += kBlock) { u += R.part[2 * c]; ke += R.part[2 * c + 1]; }
    if (R.sUs) for (long long e = R.soff_list[b] + threadIdx.x; e < R.soff_list[b + 1]; e += kBlock) u += R.sUs[e];
    u = block_sum(u, sh8); ke = block_sum(ke, sh8);
    if (threadIdx.x == 0) {
        R.out_U[b] = u; R.out_KE[b] = ke;
        if (R.out_nb) R.out_nb[b] = (long long)R.nbroken[b];
        if (!isfinite(u + ke)) atomicOr(R.flags, 1);
        if (b == 0 && R.out_step) *R.out_step = R.step;
    }
    if (R.out_R) {
        for (int g = 0; g < kMaxGroups; ++g) {
            double rx = 0.0, ry = 0.0;
            if (R.gids[g]) {   // block-uniform
                for (long long q = R.gseg[g][b] + threadIdx.x; q < R.gseg[g][b + 1]; q += kBlock) {
                    const double2 f = R.f[R.gids[g][q]];
                    rx += f.x; ry += f.y;
                }
                rx = block_sum(rx, sh8); ry = block_sum(ry, sh8);
            }
            if (threadIdx.x == 0) { R.out_R[((size_t)b * kMaxGroups + g) * 2] = rx; R.out_R[((size_t)b * kMaxGroups + g) * 2 + 1] = ry; }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Stream compaction of dead springs (a7), first half.  Gather layout: every row is compacted in place, stably (the
// summation order of the survivors is unchanged, so results are bit-identical), and the slice's live width shrinks to the
// longest surviving row; the repacking stage below then removes the freed columns from the slot storage.
// ---------------------------------------------------------------------------------------------------------------
struct CompactParams {
    TileHdr *hdr;
    int32_t *nbr, *sid;
    int16_t *nbr16;
    uint8_t *typ;
    thr_t *thr;
    double *kF, *r0F;
    long long nslices;
    uint16_t *widx;        // window indices of the windowed kernel (NULL when unused); a free slot holds the particle's own index
};

__global__ void __launch_bounds__(kBlock) k_compact_ell(const CompactParams C) {
    const long long sl = ((long long)blockIdx.x * kBlock + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (sl >= C.nslices) return;
    TileHdr *h = C.hdr + sl / kTileSlices;
    const int wi = (int)(sl % kTileSlices);
    const unsigned w = h->w[wi];
    const size_t e0 = (size_t)h->off[wi] * kSlice + lane;
    const int self = (int)(sl * kSlice + lane);
    unsigned j = 0;
    for (unsigned s = 0; s < w; ++s) {
        const size_t e = e0 + (size_t)s * kSlice;
        const int nb = C.nbr[e];
        if (nb != self) {
            if (j != s) {
                const size_t d = e0 + (size_t)j * kSlice;
                C.nbr[d] = nb; C.sid[d] = C.sid[e];
                if (C.nbr16) C.nbr16[d] = C.nbr16[e];
                if (C.widx) C.widx[d] = C.widx[e];
                if (C.typ) C.typ[d] = C.typ[e];
                if (C.thr) C.thr[d] = C.thr[e];
                if (C.kF) C.kF[d] = C.kF[e];
                if (C.r0F) C.r0F[d] = C.r0F[e];
            }
            ++j;
        }
    }
    uint16_t own_idx = 0;
    if (C.widx) { uint16_t ob; memcpy(&ob, h->pad, 2); own_idx = (uint16_t)(ob + wi * kSlice + lane); }   // TileHdr.pad[0..1] = window index of the tile's first particle
    for (unsigned s = j; s < w; ++s) {
        C.nbr[e0 + (size_t)s * kSlice] = self;
        if (C.nbr16) C.nbr16[e0 + (size_t)s * kSlice] = 0;
        if (C.widx) C.widx[e0 + (size_t)s * kSlice] = own_idx;
    }
    unsigned wmax = j;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
    if (lane == 0) h->w[wi] = (uint8_t)wmax;
}

// Repacking (second half of a7): after the in-row pass the slices' live widths have shrunk; give every slice exactly its
// live width in the slot storage, so that the streams the step kernels copy (and their byte counts: the producer sizes
// each tile's bulk copies from off[8] - off[0]) shrink with it.  Three device-only stages, no host round trip:
//   k_scan_widths   exclusive prefix sum of the live widths over all slices -> new slot offsets.  Single pass, decoupled
//                   look-back: every block publishes its aggregate, then its inclusive prefix, in one 64-bit status word
//                   (flag in the top two bits); blocks take their index from an atomic ticket so that every
//                   predecessor a block may wait for is already running.
//   k_repack_move   one warp per slice copies its live slots of one array to the new offsets in a scratch array (stable:
//                   rows keep their order, so per-particle summation order and all results are unchanged);
//   k_copy_back / k_commit_offsets   scratch -> array, then the tile headers take the new offsets.
// All stages return at once when nothing shrank (new total == old total).
struct RepackParams {
    TileHdr *hdr;
    long long nsl;                 // slices in the header table (tiles * 8)
    uint32_t *new_off;             // [nsl + 1]
    unsigned long long *state;     // [blocks] look-back status words, zeroed before the scan
    unsigned int *ticket;          // zeroed before the scan
    uint32_t *totals;              // [0] slots stored now, [1] slots after repacking
};

__global__ void __launch_bounds__(kBlock) k_scan_widths(const RepackParams R) {
    __shared__ unsigned int bid_s;
    __shared__ uint32_t wsum[kBlock / 32];
    __shared__ uint32_t excl_s;
    if (threadIdx.x == 0) bid_s = atomicAdd(R.ticket, 1u);
    __syncthreads();
    const unsigned bid = bid_s;
    const long long sl = (long long)bid * kBlock + threadIdx.x;
    const uint32_t w = sl < R.nsl ? R.hdr[sl >> 3].w[sl & 7] : 0u;
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    uint32_t x = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[wi] = x;
    __syncthreads();
    uint32_t before = 0, agg = 0;
#pragma unroll
    for (int q = 0; q < kBlock / 32; ++q) { if (q < wi) before += wsum[q]; agg += wsum[q]; }
    const uint32_t incl = before + x;
    if (threadIdx.x == 0) {
        volatile unsigned long long *st = R.state;
        uint32_t run = 0;
        if (bid > 0) {
            st[bid] = (1ull << 62) | agg;                         // aggregate available
            for (long long j = (long long)bid - 1;; --j) {        // look back until a block with its inclusive prefix
                unsigned long long v;
                do { v = st[j]; } while ((v >> 62) == 0ull);
                run += (uint32_t)v;
                if ((v >> 62) == 2ull) break;
            }
        }
        st[bid] = (2ull << 62) | (unsigned long long)(run + agg); // inclusive prefix available
        excl_s = run;
    }
    __syncthreads();
    if (sl < R.nsl) R.new_off[sl] = excl_s + incl - w;
    if (sl == R.nsl - 1) { R.new_off[R.nsl] = excl_s + incl; R.totals[1] = excl_s + incl; }
}

template <class T>
__global__ void __launch_bounds__(kBlock) k_repack_move(const RepackParams R, const T *src, T *dst) {
    if (R.totals[1] == R.totals[0]) return;
    const long long sl = ((long long)blockIdx.x * kBlock + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (sl >= R.nsl) return;
    const TileHdr *h = R.hdr + (sl >> 3);
    const unsigned w = h->w[sl & 7];
    const size_t from = (size_t)h->off[sl & 7] * kSlice + lane, to = (size_t)R.new_off[sl] * kSlice + lane;
    for (unsigned q = 0; q < w; ++q) dst[to + (size_t)q * kSlice] = src[from + (size_t)q * kSlice];
}

template <class T>
__global__ void __launch_bounds__(kBlock) k_copy_back(const RepackParams R, const T *src, T *dst) {
    if (R.totals[1] == R.totals[0]) return;
    const size_t n = (size_t)R.totals[1] * kSlice;
    for (size_t i = (size_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += (size_t)gridDim.x * kBlock) dst[i] = src[i];
}

__global__ void __launch_bounds__(kBlock) k_commit_offsets(const RepackParams R) {
    if (R.totals[1] == R.totals[0]) return;
    const long long t = (long long)blockIdx.x * kBlock + threadIdx.x;      // tile
    if (t * kTileSlices >= R.nsl) return;
    TileHdr *h = R.hdr + t;
#pragma unroll
    for (int q = 0; q <= kTileSlices; ++q) h->off[q] = R.new_off[t * kTileSlices + q];
}

__global__ void k_commit_total(uint32_t *totals) { totals[0] = totals[1]; }

// ---------------------------------------------------------------------------------------------------------------
// Per-particle virial stress, Eq. 7 without 1/Omega:  S^k = 1/2 sum_l (x^l - x^k) (x) f^kl - m v (x) v,
// f^kl = g d (Eq. 2).  One thread per particle in CALLER numbering, reading its row of the gather layout (master
// 32-bit ids; a slot holding the own id is padding or a dead spring).  IEEE sqrt / divide: this is an output pass,
// not the step.  out[c] = {S_xx, S_yy, S_xy}.
// ---------------------------------------------------------------------------------------------------------------
struct VirialParams {
    const double2 *pos, *vel;
    const uint8_t *grp;
    const double *mass;
    double mass_u, dt;
    const TileHdr *hdr;
    const int32_t *nbr;
    SpringParams sp;
    int pm;
    const int32_t *inv;   // caller id -> internal id, or NULL
    long long N;
    GroupTab g;
    double *out;          // [N][3]
};

__global__ void __launch_bounds__(kBlock) k_virial(const VirialParams V) {
    const long long c = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (c >= V.N) return;
    const int p = V.inv ? V.inv[c] : (int)c;
    const TileHdr *h = V.hdr + (p >> 8);
    const int wi = (p >> 5) & 7, lane = p & 31;
    const unsigned w = h->w[wi];
    const size_t e0 = (size_t)h->off[wi] * kSlice + lane;
    const double2 xp = V.pos[p];
    double sxx = 0.0, syy = 0.0, sxy = 0.0;
    for (unsigned s = 0; s < w; ++s) {
        const size_t e = e0 + (size_t)s * kSlice;
        const int nb = V.nbr[e];
        if (nb == p) continue;
        double k, r0;
        if (V.pm == PM_UNIFORM || V.pm == PM_RCF) { k = V.sp.k_u; r0 = V.sp.r0_u; }
        else if (V.pm == PM_TYPED || V.pm == PM_KRT_RCF) { const int t = V.sp.typ[e]; k = V.sp.tab[kTabStride * t]; r0 = V.sp.tab[kTabStride * t + 3]; }
        else { k = V.sp.kF[e]; r0 = V.sp.r0F[e]; }
        const double2 xq = V.pos[nb];
        const double dx = xq.x - xp.x, dy = xq.y - xp.y;
        const double r = sqrt(dx * dx + dy * dy);
        if (r == 0.0) continue;
        const double hg = 0.5 * (k * (r - r0) / r);
        sxx += hg * dx * dx; syy += hg * dy * dy; sxy += hg * dx * dy;
    }
    double2 v = V.vel[p];
    const uint8_t gg = V.grp[p];
    if (gg != kFree) v = make_double2(V.g.dux[gg] / V.dt, V.g.duy[gg] / V.dt);   // kinematic: the slot holds the origin
    const double m = V.mass ? V.mass[p] : V.mass_u;
    V.out[3 * c] = sxx - m * v.x * v.x;
    V.out[3 * c + 1] = syy - m * v.y * v.y;
    V.out[3 * c + 2] = sxy - m * v.x * v.y;
}

// ---------------------------------------------------------------------------------------------------------------
// Lagrangian strain field, Eq. 8, reading Q21 of DESIGN.md: per particle, the least-squares
// affine map F of the reference bond vectors d0 of its LIVE springs onto their current bond vectors d,
// F = (sum d (x) d0) (sum d0 (x) d0)^-1, eps = (F^T F - I)/2.  Particle-centric over the sliced-ELL rows (a free or dead
// slot holds the particle's own id), one thread per particle, caller order out.  POS = double2 (D = 2) or double4 (D = 3).
// Fewer than D independent reference bonds (det V <= 1e-12 (tr V / D)^D): eps = 0, ok = 0.
// ---------------------------------------------------------------------------------------------------------------
template <class POS> struct StrainParams {
    const POS *pos, *ref;     // current and reference positions, internal numbering
    const TileHdr *hdr;
    const int32_t *nbr;
    const int32_t *inv;       // caller id -> internal id, or NULL
    long long N;
    double *out;              // [N][3] {xx, yy, xy} or [N][6] {xx, yy, zz, xy, yz, zx}
    uint8_t *ok;              // [N]
};

__global__ void __launch_bounds__(kBlock) k_strain2(const StrainParams<double2> S) {
    const long long c = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (c >= S.N) return;
    const int p = S.inv ? S.inv[c] : (int)c;
    const TileHdr *h = S.hdr + (p >> 8);
    const int wi = (p >> 5) & 7, lane = p & 31;
    const unsigned w = h->w[wi];
    const size_t e0 = (size_t)h->off[wi] * kSlice + lane;
    const double2 xp = S.pos[p], rp = S.ref[p];
    double vxx = 0.0, vxy = 0.0, vyy = 0.0, wxx = 0.0, wxy = 0.0, wyx = 0.0, wyy = 0.0;
    for (unsigned s = 0; s < w; ++s) {
        const int nb = S.nbr[e0 + (size_t)s * kSlice];
        if (nb == p) continue;
        const double2 xq = S.pos[nb], rq = S.ref[nb];
        const double ax = rq.x - rp.x, ay = rq.y - rp.y, dx = xq.x - xp.x, dy = xq.y - xp.y;
        vxx += ax * ax; vxy += ax * ay; vyy += ay * ay;
        wxx += dx * ax; wxy += dx * ay; wyx += dy * ax; wyy += dy * ay;     // W = sum d (x) d0
    }
    const double det = vxx * vyy - vxy * vxy, tr = 0.5 * (vxx + vyy);
    double exx = 0.0, eyy = 0.0, exy = 0.0;
    const bool good = det > 1e-12 * tr * tr;
    if (good) {
        const double ixx = vyy / det, ixy = -vxy / det, iyy = vxx / det;
        const double fxx = wxx * ixx + wxy * ixy, fxy = wxx * ixy + wxy * iyy, fyx = wyx * ixx + wyy * ixy, fyy = wyx * ixy + wyy * iyy;
        exx = 0.5 * (fxx * fxx + fyx * fyx - 1.0);
        eyy = 0.5 * (fxy * fxy + fyy * fyy - 1.0);
        exy = 0.5 * (fxx * fxy + fyx * fyy);
    }
    S.out[3 * c] = exx; S.out[3 * c + 1] = eyy; S.out[3 * c + 2] = exy;
    S.ok[c] = good ? 1 : 0;
}

__global__ void __launch_bounds__(kBlock) k_strain3(const StrainParams<double4> S) {
    const long long c = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (c >= S.N) return;
    const int p = S.inv ? S.inv[c] : (int)c;
    const TileHdr *h = S.hdr + (p >> 8);
    const int wi = (p >> 5) & 7, lane = p & 31;
    const unsigned w = h->w[wi];
    const size_t e0 = (size_t)h->off[wi] * kSlice + lane;
    const double4 xp = S.pos[p], rp = S.ref[p];
    double v[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};      // xx xy xz yy yz zz
    double m[9] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};   // W row-major
    for (unsigned s = 0; s < w; ++s) {
        const int nb = S.nbr[e0 + (size_t)s * kSlice];
        if (nb == p) continue;
        const double4 xq = S.pos[nb], rq = S.ref[nb];
        const double a[3] = {rq.x - rp.x, rq.y - rp.y, rq.z - rp.z}, d[3] = {xq.x - xp.x, xq.y - xp.y, xq.z - xp.z};
        v[0] += a[0] * a[0]; v[1] += a[0] * a[1]; v[2] += a[0] * a[2]; v[3] += a[1] * a[1]; v[4] += a[1] * a[2]; v[5] += a[2] * a[2];
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) m[3 * i + j] += d[i] * a[j];
    }
    // cofactors of the symmetric V
    const double c00 = v[3] * v[5] - v[4] * v[4], c01 = v[4] * v[2] - v[1] * v[5], c02 = v[1] * v[4] - v[3] * v[2];
    const double det = v[0] * c00 + v[1] * c01 + v[2] * c02, tr = (v[0] + v[3] + v[5]) / 3.0;
    double e[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    const bool good = det > 1e-12 * tr * tr * tr;
    if (good) {
        double iv[9];
        iv[0] = c00 / det; iv[1] = c01 / det; iv[2] = c02 / det;
        iv[3] = iv[1]; iv[4] = (v[0] * v[5] - v[2] * v[2]) / det; iv[5] = (v[2] * v[1] - v[0] * v[4]) / det;
        iv[6] = iv[2]; iv[7] = iv[5]; iv[8] = (v[0] * v[3] - v[1] * v[1]) / det;
        double F[9];
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) F[3 * i + j] = m[3 * i] * iv[j] + m[3 * i + 1] * iv[3 + j] + m[3 * i + 2] * iv[6 + j];
        auto ftf = [&](int a, int b) { return F[a] * F[b] + F[3 + a] * F[3 + b] + F[6 + a] * F[6 + b]; };
        e[0] = 0.5 * (ftf(0, 0) - 1.0); e[1] = 0.5 * (ftf(1, 1) - 1.0); e[2] = 0.5 * (ftf(2, 2) - 1.0);
        e[3] = 0.5 * ftf(0, 1); e[4] = 0.5 * ftf(1, 2); e[5] = 0.5 * ftf(2, 0);
    }
#pragma unroll
    for (int q = 0; q < 6; ++q) S.out[6 * c + q] = e[q];
    S.ok[c] = good ? 1 : 0;
}

// ---- small utility kernels (numbering translation at the API boundary, boundary-group bookkeeping) ----
// dst[perm_dst[q]] <- src[q] style copies.  inv: caller id -> internal id.
__global__ void __launch_bounds__(kBlock) k_to_caller(const double2 *src, double2 *dst, const int32_t *inv, long long N,
                                                      const uint8_t *grp, GroupTab g, double dt, int synth_vel) {
    const long long c = (long long)blockIdx.x * kBlock + threadIdx.x;  // caller id
    if (c >= N) return;
    const int p = inv ? inv[c] : (int)c;
    double2 v = src[p];
    if (synth_vel) { const uint8_t gg = grp[p]; if (gg != kFree) v = make_double2(g.dux[gg] / dt, g.duy[gg] / dt); }
    dst[c] = v;
}

// Input validation of lsm_write_state on the device (the staged copies of the caller's arrays): *bad |= 1 on NaN / Inf.
__global__ void __launch_bounds__(kBlock) k_check_finite(const double *a, const double *b, long long n, int *bad) {
    bool ok = true;
    for (long long q = (long long)blockIdx.x * kBlock + threadIdx.x; q < n; q += (long long)gridDim.x * kBlock)
        ok = ok && isfinite(a[q]) && (!b || isfinite(b[q]));
    if (!ok) atomicOr(bad, 1);
}

__global__ void __launch_bounds__(kBlock) k_from_caller(const double2 *srcx, const double2 *srcv, double2 *pos, double2 *vel,
                                                        const int32_t *inv, long long N, const uint8_t *grp) {
    const long long c = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (c >= N) return;
    const int p = inv ? inv[c] : (int)c;
    const double2 x = srcx[c];
    pos[p] = x;
    vel[p] = (grp[p] != kFree) ? x : (srcv ? srcv[c] : make_double2(0.0, 0.0));  // kinematic: vel slot = origin
}

// Released particles become free with the kinematic velocity (vx, vy) = du/dt they were carrying; their kinetic-energy
// term (kept per particle for lsm_read_energy) follows.  Nothing else changes: f and the held fd stay (R3).
__global__ void __launch_bounds__(kBlock) k_group_release(const int32_t *ids, long long n, uint8_t *grp, double2 *vel, double vx, double vy,
                                                          double *sKE, const double *mass, double mass_u) {
    const long long q = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (q >= n) return;
    const int p = ids[q];
    grp[p] = kFree;
    vel[p] = make_double2(vx, vy);
    const double m = mass ? mass[p] : mass_u;
    sKE[p] = __dmul_rn(__dmul_rn(0.5, m), __dadd_rn(__dmul_rn(vx, vx), __dmul_rn(vy, vy)));
}

__global__ void __launch_bounds__(kBlock) k_group_assign(const int32_t *ids, long long n, uint8_t *grp, double2 *vel, const double2 *pos, uint8_t g,
                                                         double *sKE) {
    const long long q = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (q >= n) return;
    const int p = ids[q];
    grp[p] = g;
    vel[p] = pos[p];        // kinematic: the vel slot holds the origin
    sKE[p] = 0.0;           // kinematic particles carry no KE (Q6)
}

// Velocity ramp of the strain-rate protocol (lsm_set_strain_rate): every free particle takes, along `axis`, the velocity
// of the affine field that moves the grips apart, v = e (x - c) / dt (e = strain per step, c = the fixed point).
// One coordinate of the listed particles (internal ids), in list order: the gauge-length means of lsm_set_strain_rate.
__global__ void __launch_bounds__(kBlock) k_gather_axis(const double2 *pos, const int32_t *ids, long long n, int axis, double *out) {
    const long long q = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (q < n) { const double2 r = pos[ids[q]]; out[q] = axis == 0 ? r.x : r.y; }
}

__global__ void __launch_bounds__(kBlock) k_velocity_ramp(const double2 *pos, double2 *vel, const uint8_t *grp, long long N, int axis, double e, double c, double dt) {
    const long long p = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (p >= N || grp[p] != kFree) return;
    const double2 x = pos[p];
    double2 v = vel[p];
    const double r = __ddiv_rn(__dmul_rn(e, __dsub_rn(axis == 0 ? x.x : x.y, c)), dt);
    if (axis == 0) v.x = r; else v.y = r;
    vel[p] = v;
}

__global__ void __launch_bounds__(kBlock) k_broken_from_steps(const long long *break_step, uint8_t *broken, long long M) {
    const long long e = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (e < M) broken[e] = break_step[e] >= 0;
}

}  // namespace lsmk
