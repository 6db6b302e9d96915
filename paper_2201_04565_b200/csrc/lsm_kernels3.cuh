// lsm_kernels3.cuh -- the D = 3 path (the paper's own array layout is 3-D: kernel listing PAPER.md:L93-L97, "larger and
// three-dimensional models" L198).  A first, plain version of the same fused gather step as lsm_kernels.cuh: one thread
// per particle, every stream read straight from global memory, no shared-memory pipeline, IEEE sqrt / divide in both
// arithmetic modes.  It reuses the sliced-ELL spring layout, the breakage bookkeeping, the chunk reductions and the
// compaction of the 2-D path unchanged; only the particle state differs:
//   pos3[2][Npad], vel3[Npad], f3[N], fd3[N]   double4 {x, y, z, 0}: one aligned 32-byte record per particle.
// Every 2-D configuration of BASELINE.json runs on the tuned 2-D kernels; this path is correctness-first (parity-tested
// against the oracle, bit-identical in exact mode) and its speed is reported as measured, not tuned.
#pragma once
#include "lsm_kernels.cuh"

namespace lsmk {

struct GroupTab3 {
    double du[3][kMaxGroups];
    long long n0[kMaxGroups];
};

struct Step3Params {
    const double4 *pos_cur;
    double4 *pos_next;
    double4 *vel, *f, *fd;
    const uint8_t *grp;
    const double *mass;
    double mass_u, dt, hdt, gamma;
    long long N, step;
    const TileHdr *hdr;
    int32_t *nbr;
    int16_t *nbr16;      // kept consistent for compaction; not read here
    const int32_t *sid;
    SpringParams sp;
    int pm;
    long long *break_step;
    unsigned long long *nbroken;
    const long long *poff;
    int B;
    double *sU, *sKE;
    int kick2, advance, sample;
    GroupTab3 g;
};

// One launch = force evaluation at the current positions (+ breakage), damping, second half kick, and (advance) the
// first half kick + drift of the next step: the same order and the same rounding sequence as particle_update / the
// serial reference loop.  EXACT: never-contracted arithmetic; !EXACT: the compiler may fuse multiply-adds.
template <bool EXACT>
__global__ void __launch_bounds__(kBlock) k3_step(const Step3Params P) {
    const long long p = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (p >= P.N) return;
    const TileHdr *h = P.hdr + (p >> 8);
    const int wi = (int)(p >> 5) & 7, lane = (int)p & 31;
    const unsigned w = h->w[wi];
    const size_t e0 = (size_t)h->off[wi] * kSlice + lane;
    const double4 xp = P.pos_cur[p];
    double fx = 0.0, fy = 0.0, fz = 0.0, u = 0.0;
    for (unsigned s = 0; s < w; ++s) {
        const size_t e = e0 + (size_t)s * kSlice;
        const int nb = P.nbr[e];
        if (nb == (int)p) continue;                              // padding or dead spring
        double k, r0, rc;
        if (P.pm == PM_UNIFORM) { k = P.sp.k_u; r0 = P.sp.r0_u; rc = P.sp.rc_u; }
        else if (P.pm == PM_TYPED) { const int t = P.sp.typ[e]; k = P.sp.tab[kTabStride * t]; r0 = P.sp.tab[kTabStride * t + 3]; rc = P.sp.tab[kTabStride * t + 4]; }
        else if (P.pm == PM_RCF) { k = P.sp.k_u; r0 = P.sp.r0_u; rc = P.sp.rcS[P.sid[e]]; }
        else if (P.pm == PM_KRT_RCF) { const int t = P.sp.typ[e]; k = P.sp.tab[kTabStride * t]; r0 = P.sp.tab[kTabStride * t + 3]; rc = P.sp.rcS[P.sid[e]]; }
        else { k = P.sp.kF[e]; r0 = P.sp.r0F[e]; rc = P.sp.rcS[P.sid[e]]; }
        const double4 xq = P.pos_cur[nb];
        const double dx = sub<EXACT>(xq.x, xp.x), dy = sub<EXACT>(xq.y, xp.y), dz = sub<EXACT>(xq.z, xp.z);
        // r2 accumulated component by component from 0 like the oracle ((dx^2 + dy^2) + dz^2)
        const double r2 = add<EXACT>(add<EXACT>(mul<EXACT>(dx, dx), mul<EXACT>(dy, dy)), mul<EXACT>(dz, dz));
        const double r = __dsqrt_rn(r2);
        if (r > rc) {                                            // strict '>' (Q1); irreversible (Q2); no force now (Q3)
            P.nbr[e] = (int)p;
            if (P.nbr16) P.nbr16[e] = 0;
            if (p < nb) {
                P.break_step[P.sid[e]] = P.step;
                atomicAdd(P.nbroken + spec_of(P.poff, P.B, p), 1ULL);
            }
            continue;
        }
        if (r == 0.0) continue;                                  // coincident endpoints (Q4)
        const double ext = sub<EXACT>(r, r0);
        const double g = __ddiv_rn(mul<EXACT>(k, ext), r);
        fx = mad<EXACT>(g, dx, fx); fy = mad<EXACT>(g, dy, fy); fz = mad<EXACT>(g, dz, fz);
        if (P.sample && p < nb) u = add<EXACT>(u, mul<EXACT>(mul<EXACT>(mul<EXACT>(0.5, k), ext), ext));
    }
    const double4 vh = P.vel[p];
    const uint8_t gg = P.grp[p];
    if (gg == kFree) {
        const double fdx = sub<EXACT>(fx, mul<EXACT>(P.gamma, vh.x)), fdy = sub<EXACT>(fy, mul<EXACT>(P.gamma, vh.y)),
                     fdz = sub<EXACT>(fz, mul<EXACT>(P.gamma, vh.z));
        const double m = P.mass ? P.mass[p] : P.mass_u;
        const double ax = __ddiv_rn(fdx, m), ay = __ddiv_rn(fdy, m), az = __ddiv_rn(fdz, m);
        double4 v = vh;
        if (P.kick2) { v.x = mad<EXACT>(P.hdt, ax, vh.x); v.y = mad<EXACT>(P.hdt, ay, vh.y); v.z = mad<EXACT>(P.hdt, az, vh.z); }
        if (P.sample) {
            const double v2 = add<EXACT>(add<EXACT>(mul<EXACT>(v.x, v.x), mul<EXACT>(v.y, v.y)), mul<EXACT>(v.z, v.z));
            P.sU[p] = u;
            P.sKE[p] = mul<EXACT>(mul<EXACT>(0.5, m), v2);
        }
        if (P.sample || !P.advance) P.f[p] = make_double4(fx, fy, fz, 0.0);
        if (P.advance) {
            double4 wv, xn;
            wv.x = mad<EXACT>(P.hdt, ax, v.x); wv.y = mad<EXACT>(P.hdt, ay, v.y); wv.z = mad<EXACT>(P.hdt, az, v.z); wv.w = 0.0;
            xn.x = mad<EXACT>(P.dt, wv.x, xp.x); xn.y = mad<EXACT>(P.dt, wv.y, xp.y); xn.z = mad<EXACT>(P.dt, wv.z, xp.z); xn.w = 0.0;
            P.pos_next[p] = xn;
            P.vel[p] = wv;
        } else {
            P.vel[p] = v;
            P.fd[p] = make_double4(fdx, fdy, fdz, 0.0);
        }
    } else {  // kinematic: vh holds the origin
        if (P.sample) { P.sU[p] = u; P.sKE[p] = 0.0; }
        if (P.sample || !P.advance) P.f[p] = make_double4(fx, fy, fz, 0.0);
        if (P.advance) {
            const double ns = (double)(P.step + 1 - P.g.n0[gg]);
            P.pos_next[p] = make_double4(mad<EXACT>(ns, P.g.du[0][gg], vh.x), mad<EXACT>(ns, P.g.du[1][gg], vh.y),
                                         mad<EXACT>(ns, P.g.du[2][gg], vh.z), 0.0);
        } else {   // held total force of a kinematic particle: f - gamma * (du/dt) (see particle_update)
            const double vkx = __ddiv_rn(P.g.du[0][gg], P.dt), vky = __ddiv_rn(P.g.du[1][gg], P.dt), vkz = __ddiv_rn(P.g.du[2][gg], P.dt);
            P.fd[p] = make_double4(sub<EXACT>(fx, mul<EXACT>(P.gamma, vkx)), sub<EXACT>(fy, mul<EXACT>(P.gamma, vky)),
                                   sub<EXACT>(fz, mul<EXACT>(P.gamma, vkz)), 0.0);
        }
    }
}

// First half kick + drift from a completed state (v, fd): the first kernel of every lsm_step call.
template <bool EXACT>
__global__ void __launch_bounds__(kBlock) k3_start(const Step3Params P) {
    const long long p = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (p >= P.N) return;
    const double4 xp = P.pos_cur[p], v = P.vel[p];
    const uint8_t gg = P.grp[p];
    if (gg == kFree) {
        const double4 fd = P.fd[p];
        const double m = P.mass ? P.mass[p] : P.mass_u;
        const double ax = __ddiv_rn(fd.x, m), ay = __ddiv_rn(fd.y, m), az = __ddiv_rn(fd.z, m);
        double4 wv, xn;
        wv.x = mad<EXACT>(P.hdt, ax, v.x); wv.y = mad<EXACT>(P.hdt, ay, v.y); wv.z = mad<EXACT>(P.hdt, az, v.z); wv.w = 0.0;
        xn.x = mad<EXACT>(P.dt, wv.x, xp.x); xn.y = mad<EXACT>(P.dt, wv.y, xp.y); xn.z = mad<EXACT>(P.dt, wv.z, xp.z); xn.w = 0.0;
        P.pos_next[p] = xn;
        P.vel[p] = wv;
    } else {
        const double ns = (double)(P.step + 1 - P.g.n0[gg]);
        P.pos_next[p] = make_double4(mad<EXACT>(ns, P.g.du[0][gg], v.x), mad<EXACT>(ns, P.g.du[1][gg], v.y),
                                     mad<EXACT>(ns, P.g.du[2][gg], v.z), 0.0);
    }
}

// Sample finalisation with 3-component reactions: same fixed-order block sums as k_finalize_sample.
struct Reduce3Params {
    ReduceParams R;        // chunk partials, outputs for U / KE / n_broken / step (R.f and R.out_R unused)
    const double4 *f3;
    double *out_R3;        // [B][8][3] or NULL
};

__global__ void __launch_bounds__(kBlock) k3_finalize_sample(const Reduce3Params Q) {
    __shared__ double sh8[kBlock / 32];
    const ReduceParams &R = Q.R;
    const int b = blockIdx.x;
    double u = 0.0, ke = 0.0;
    for (int c = R.spec_chunk_off[b] + threadIdx.x; c < R.spec_chunk_off[b + 1]; c += kBlock) { u += R.part[2 * c]; ke += R.part[2 * c + 1]; }
    u = block_sum(u, sh8); ke = block_sum(ke, sh8);
    if (threadIdx.x == 0) {
        R.out_U[b] = u; R.out_KE[b] = ke;
        if (R.out_nb) R.out_nb[b] = (long long)R.nbroken[b];
        if (!isfinite(u + ke)) atomicOr(R.flags, 1);
        if (b == 0 && R.out_step) *R.out_step = R.step;
    }
    if (Q.out_R3) {
        for (int g = 0; g < kMaxGroups; ++g) {
            double rx = 0.0, ry = 0.0, rz = 0.0;
            if (R.gids[g]) {
                for (long long q = R.gseg[g][b] + threadIdx.x; q < R.gseg[g][b + 1]; q += kBlock) {
                    const double4 f = Q.f3[R.gids[g][q]];
                    rx += f.x; ry += f.y; rz += f.z;
                }
                rx = block_sum(rx, sh8); ry = block_sum(ry, sh8); rz = block_sum(rz, sh8);
            }
            if (threadIdx.x == 0) {
                double *o = Q.out_R3 + ((size_t)b * kMaxGroups + g) * 3;
                o[0] = rx; o[1] = ry; o[2] = rz;
            }
        }
    }
}

// Per-particle virial stress in 3-D (Eq. 7, without 1/Omega): out[c] = {S_xx, S_yy, S_zz, S_xy, S_yz, S_zx}.
// Same structure as k_virial (one thread per particle in caller numbering, master 32-bit ids, IEEE sqrt / divide).
struct Virial3Params {
    const double4 *pos, *vel;
    const uint8_t *grp;
    const double *mass;
    double mass_u, dt;
    const TileHdr *hdr;
    const int32_t *nbr;
    SpringParams sp;
    int pm;
    const int32_t *inv;
    long long N;
    GroupTab3 g;
    double *out;          // [N][6]
};

__global__ void __launch_bounds__(kBlock) k3_virial(const Virial3Params V) {
    const long long c = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (c >= V.N) return;
    const int p = V.inv ? V.inv[c] : (int)c;
    const TileHdr *h = V.hdr + (p >> 8);
    const int wi = (p >> 5) & 7, lane = p & 31;
    const unsigned w = h->w[wi];
    const size_t e0 = (size_t)h->off[wi] * kSlice + lane;
    const double4 xp = V.pos[p];
    double s[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (unsigned q = 0; q < w; ++q) {
        const size_t e = e0 + (size_t)q * kSlice;
        const int nb = V.nbr[e];
        if (nb == p) continue;
        double k, r0;
        if (V.pm == PM_UNIFORM || V.pm == PM_RCF) { k = V.sp.k_u; r0 = V.sp.r0_u; }
        else if (V.pm == PM_TYPED || V.pm == PM_KRT_RCF) { const int t = V.sp.typ[e]; k = V.sp.tab[kTabStride * t]; r0 = V.sp.tab[kTabStride * t + 3]; }
        else { k = V.sp.kF[e]; r0 = V.sp.r0F[e]; }
        const double4 xq = V.pos[nb];
        const double dx = xq.x - xp.x, dy = xq.y - xp.y, dz = xq.z - xp.z;
        const double r = sqrt(dx * dx + dy * dy + dz * dz);
        if (r == 0.0) continue;
        const double hg = 0.5 * (k * (r - r0) / r);
        s[0] += hg * dx * dx; s[1] += hg * dy * dy; s[2] += hg * dz * dz;
        s[3] += hg * dx * dy; s[4] += hg * dy * dz; s[5] += hg * dz * dx;
    }
    double4 v = V.vel[p];
    const uint8_t gg = V.grp[p];
    if (gg != kFree) v = make_double4(V.g.du[0][gg] / V.dt, V.g.du[1][gg] / V.dt, V.g.du[2][gg] / V.dt, 0.0);
    const double m = V.mass ? V.mass[p] : V.mass_u;
    double *o = V.out + 6 * c;
    o[0] = s[0] - m * v.x * v.x; o[1] = s[1] - m * v.y * v.y; o[2] = s[2] - m * v.z * v.z;
    o[3] = s[3] - m * v.x * v.y; o[4] = s[4] - m * v.y * v.z; o[5] = s[5] - m * v.z * v.x;
}

// Numbering translation at the boundary: packed [N*3] caller arrays <-> double4 internal arrays.
__global__ void __launch_bounds__(kBlock) k3_to_caller(const double4 *src, double *dst, const int32_t *inv, long long N,
                                                       const uint8_t *grp, GroupTab3 g, double dt, int synth_vel) {
    const long long c = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (c >= N) return;
    const int p = inv ? inv[c] : (int)c;
    double4 v = src[p];
    if (synth_vel) { const uint8_t gg = grp[p]; if (gg != kFree) v = make_double4(g.du[0][gg] / dt, g.du[1][gg] / dt, g.du[2][gg] / dt, 0.0); }
    dst[3 * c] = v.x; dst[3 * c + 1] = v.y; dst[3 * c + 2] = v.z;
}

__global__ void __launch_bounds__(kBlock) k3_from_caller(const double *srcx, const double *srcv, double4 *pos, double4 *vel,
                                                         const int32_t *inv, long long N, const uint8_t *grp) {
    const long long c = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (c >= N) return;
    const int p = inv ? inv[c] : (int)c;
    const double4 x = make_double4(srcx[3 * c], srcx[3 * c + 1], srcx[3 * c + 2], 0.0);
    pos[p] = x;
    vel[p] = (grp[p] != kFree) ? x : (srcv ? make_double4(srcv[3 * c], srcv[3 * c + 1], srcv[3 * c + 2], 0.0) : make_double4(0.0, 0.0, 0.0, 0.0));
}

__global__ void __launch_bounds__(kBlock) k3_group_release(const int32_t *ids, long long n, uint8_t *grp, double4 *vel, double vx, double vy, double vz,
                                                           double *sKE, const double *mass, double mass_u) {
    const long long q = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (q >= n) return;
    const int p = ids[q];
    grp[p] = kFree;
    vel[p] = make_double4(vx, vy, vz, 0.0);
    const double m = mass ? mass[p] : mass_u;
    sKE[p] = __dmul_rn(__dmul_rn(0.5, m), __dadd_rn(__dadd_rn(__dmul_rn(vx, vx), __dmul_rn(vy, vy)), __dmul_rn(vz, vz)));
}

__global__ void __launch_bounds__(kBlock) k3_group_assign(const int32_t *ids, long long n, uint8_t *grp, double4 *vel, const double4 *pos, uint8_t g,
                                                          double *sKE) {
    const long long q = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (q >= n) return;
    const int p = ids[q];
    grp[p] = g;
    vel[p] = pos[p];
    sKE[p] = 0.0;
}

}  // namespace lsmk
