// lsm_rows3.cuh -- D = 3 row evaluation and particle update for the streamed kernel (k_gather_stream<..., D = 3>):
// the same two-pass scheme, breakage filter and arithmetic as the 2-D functions of lsm_kernels.cuh, with a z component.
// Included from lsm_kernels.cuh (it needs StepParams, RowSrc, slot_params, rsqrt_fast, ...).  In the D = 3 instantiation
// the position / velocity pointers of StepParams and StepVar address double4 {x, y, z, 0} records.
#pragma once

namespace lsmk {

__device__ __forceinline__ const double4 *as4(const double2 *p) { return reinterpret_cast<const double4 *>(p); }
__device__ __forceinline__ double4 *as4(double2 *p) { return reinterpret_cast<double4 *>(p); }

template <bool COHERENT> __device__ __forceinline__ double4 load_pos3(const double4 *p) {
    // two 16-byte halves of one aligned 32-byte record (same sector)
    const double2 *q = reinterpret_cast<const double2 *>(p);
    const double2 a = COHERENT ? __ldcg(q) : __ldg(q);
    const double2 b = COHERENT ? __ldcg(q + 1) : __ldg(q + 1);
    return make_double4(a.x, a.y, b.x, 0.0);
}

// One spring seen from one endpoint, 3-D (see slot_eval).  EXACT: r2 = ((dx^2 + dy^2) + dz^2), never contracted.
template <bool EXACT, bool SAMPLE>
__device__ __forceinline__ void slot_eval3(double4 xq, double4 xp, bool lower, double k, double r0, double kr0, uint32_t thr,
                                           double &dx, double &dy, double &dz, double &r2, double &g, double &ue, bool &near) {
    dx = sub<EXACT>(xq.x, xp.x); dy = sub<EXACT>(xq.y, xp.y); dz = sub<EXACT>(xq.z, xp.z);
    r2 = EXACT ? add<true>(add<true>(mul<true>(dx, dx), mul<true>(dy, dy)), mul<true>(dz, dz))
               : fma(dz, dz, fma(dy, dy, fma(dx, dx, 1e-300)));
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
        g = fma(-kr0, rinv, k);
        if (SAMPLE) { const double ext = fma(r2, rinv, -r0); ue = (0.5 * k) * ext * ext; }
        live = r2 > 1e-290;
    }
    if (EXACT) g = live ? g : 0.0;
    if (SAMPLE) ue = (live && lower) ? ue : 0.0;
    near = EXACT ? (live && hi >= thr) : (hi >= thr);
}

template <int PM, bool EXACT, bool SAMPLE, bool COHERENT, bool I16, int CH>
__device__ __forceinline__ bool row_chunk3(const StepParams &P, const StepVar &V, const RowSrc &R, const double *s_tab, int p, unsigned s0,
                                           double4 xp, double &fx, double &fy, double &fz, double &u) {
    int nb[CH];
    double4 xq[CH];
    bool any_near = false;
    const double4 *own = as4(V.pos_cur) + p;
    asm("" : "+l"(own));   // as in row_chunk: one wide multiply-add per gather address
#pragma unroll
    for (int c = 0; c < CH; ++c) nb[c] = I16 ? (int)R.nbr16[(s0 + c) * kSlice] : R.nbr[(s0 + c) * kSlice];
#pragma unroll
    for (int c = 0; c < CH; ++c) {
        xq[c] = I16 ? load_pos3<COHERENT>(own + nb[c]) : load_pos3<COHERENT>(as4(V.pos_cur) + nb[c]);
        if (I16) nb[c] += p;
    }
#pragma unroll
    for (int c = 0; c < CH; ++c) {
        double k, r0, kr0, dx, dy, dz, r2, g, ue;
        uint32_t thr;
        bool near;
        slot_params<PM>(P, R, s_tab, (s0 + c) * kSlice, k, r0, kr0, thr);
        slot_eval3<EXACT, SAMPLE>(xq[c], xp, p < nb[c], k, r0, kr0, thr, dx, dy, dz, r2, g, ue, near);
        fx = mad<EXACT>(g, dx, fx); fy = mad<EXACT>(g, dy, fy); fz = mad<EXACT>(g, dz, fz);
        if (SAMPLE) u = add<EXACT>(u, ue);
        any_near |= near;
    }
    return any_near;
}

template <int PM, bool EXACT, bool SAMPLE, bool COHERENT, bool I16>
__device__ __forceinline__ void row_careful3(const StepParams &P, const StepVar &V, const RowSrc &R, const double *s_tab, int p, unsigned w,
                                             double4 xp, double &fx, double &fy, double &fz, double &u) {
    fx = 0.0; fy = 0.0; fz = 0.0; u = 0.0;
#pragma unroll 1
    for (unsigned s = 0; s < w; ++s) {
        const unsigned so = s * kSlice;
        const int nb = I16 ? p + (int)R.nbr16[so] : R.nbr[so];
        const double4 xq = load_pos3<COHERENT>(as4(V.pos_cur) + nb);
        double k, r0, kr0, dx, dy, dz, r2, g, ue;
        uint32_t thr;
        bool near;
        slot_params<PM>(P, R, s_tab, so, k, r0, kr0, thr);
        slot_eval3<EXACT, SAMPLE>(xq, xp, p < nb, k, r0, kr0, thr, dx, dy, dz, r2, g, ue, near);
        if (near) {
            const size_t e = R.e0 + so;
            double rc;
            if (PM == PM_UNIFORM) rc = P.sp.rc_u;
            else if (PM == PM_TYPED) rc = s_tab[kTabStride * R.typ[so] + 4];
            else rc = __ldg(P.sp.rcS + __ldg(P.sid + e));
            if (__dsqrt_rn(r2) > rc) {   // strict '>' (Q1)
                P.nbr[e] = p;
                if (P.nbr16) P.nbr16[e] = 0;
                if (I16) const_cast<int16_t *>(R.nbr16)[so] = 0;
                else const_cast<int32_t *>(R.nbr)[so] = p;
                if (p < nb) {
                    P.break_step[P.sid[e]] = V.step;
                    atomicAdd(P.nbroken + spec_of(P.poff, P.B, p), 1ULL);
                }
                continue;
            }
        }
        fx = mad<EXACT>(g, dx, fx); fy = mad<EXACT>(g, dy, fy); fz = mad<EXACT>(g, dz, fz);
        if (SAMPLE) u = add<EXACT>(u, ue);
    }
}

template <int PM, bool EXACT, bool SAMPLE, bool COHERENT, bool I16>
__device__ __forceinline__ void row_forces3(const StepParams &P, const StepVar &V, const RowSrc &R, const double *s_tab, int p, unsigned w,
                                            double4 xp, double &fx, double &fy, double &fz, double &u) {
    constexpr int CH = kRowCH3;
    unsigned s0 = 0;
    bool any_near = false;
    for (; s0 + CH <= w; s0 += CH) any_near |= row_chunk3<PM, EXACT, SAMPLE, COHERENT, I16, CH>(P, V, R, s_tab, p, s0, xp, fx, fy, fz, u);
    for (; s0 < w; ++s0) any_near |= row_chunk3<PM, EXACT, SAMPLE, COHERENT, I16, 1>(P, V, R, s_tab, p, s0, xp, fx, fy, fz, u);
    if (any_near) row_careful3<PM, EXACT, SAMPLE, COHERENT, I16>(P, V, R, s_tab, p, w, xp, fx, fy, fz, u);
}

// Velocity-Verlet particle update in 3-D (see particle_update): same order, same rounding sequence.
template <bool EXACT, bool KICK2, bool ADVANCE, bool SAMPLE>
__device__ __forceinline__ void particle_update3(const StepParams &P, const StepVar &V, long long p, double4 xp, double4 vh, uint8_t g,
                                                 double fx, double fy, double fz, double u, double4 *own_pos = nullptr, double4 *own_vel = nullptr) {
    double4 *pos_next = as4(V.pos_next), *vel = as4(P.vel), *f = as4(P.f), *fd = as4(P.fd);
    if (g == kFree) {
        const double fdx = sub<EXACT>(fx, mul<EXACT>(P.gamma, vh.x)), fdy = sub<EXACT>(fy, mul<EXACT>(P.gamma, vh.y)),
                     fdz = sub<EXACT>(fz, mul<EXACT>(P.gamma, vh.z));
        double ax, ay, az, m;
        if (P.mass) { m = __ldg(P.mass + p); ax = __ddiv_rn(fdx, m); ay = __ddiv_rn(fdy, m); az = __ddiv_rn(fdz, m); }
        else if (EXACT) { m = P.mass_u; ax = __ddiv_rn(fdx, m); ay = __ddiv_rn(fdy, m); az = __ddiv_rn(fdz, m); }
        else { m = P.mass_u; ax = fdx * P.inv_mass_u; ay = fdy * P.inv_mass_u; az = fdz * P.inv_mass_u; }
        double4 v = vh;
        if (KICK2) { v.x = mad<EXACT>(P.hdt, ax, vh.x); v.y = mad<EXACT>(P.hdt, ay, vh.y); v.z = mad<EXACT>(P.hdt, az, vh.z); }
        if (SAMPLE) {
            const double v2 = add<EXACT>(add<EXACT>(mul<EXACT>(v.x, v.x), mul<EXACT>(v.y, v.y)), mul<EXACT>(v.z, v.z));
            P.sU[p] = u;
            P.sKE[p] = mul<EXACT>(mul<EXACT>(0.5, m), v2);
        }
        if (SAMPLE || !ADVANCE) f[p] = make_double4(fx, fy, fz, 0.0);
        if (ADVANCE) {
            double4 w, xn;
            if (!EXACT && KICK2 && !SAMPLE) { w.x = fma(P.dt, ax, vh.x); w.y = fma(P.dt, ay, vh.y); w.z = fma(P.dt, az, vh.z); }
            else { w.x = mad<EXACT>(P.hdt, ax, v.x); w.y = mad<EXACT>(P.hdt, ay, v.y); w.z = mad<EXACT>(P.hdt, az, v.z); }
            w.w = 0.0;
            xn.x = mad<EXACT>(P.dt, w.x, xp.x); xn.y = mad<EXACT>(P.dt, w.y, xp.y); xn.z = mad<EXACT>(P.dt, w.z, xp.z); xn.w = 0.0;
            pos_next[p] = xn;
            vel[p] = w;
            if (own_pos) { *own_pos = xn; *own_vel = w; }   // resident tiles: the staged copy is the next step's input
        } else {
            vel[p] = v;
            fd[p] = make_double4(fdx, fdy, fdz, 0.0);
        }
    } else {  // kinematic: vh holds the origin
        if (SAMPLE) { P.sU[p] = u; P.sKE[p] = 0.0; }
        if (SAMPLE || !ADVANCE) f[p] = make_double4(fx, fy, fz, 0.0);
        if (ADVANCE) {
            const double ns = (double)(V.step + 1 - P.g.n0[g]);
            const double4 xn = make_double4(mad<EXACT>(ns, P.g.dux[g], vh.x), mad<EXACT>(ns, P.g.duy[g], vh.y), mad<EXACT>(ns, P.g.duz[g], vh.z), 0.0);
            pos_next[p] = xn;
            if (own_pos) *own_pos = xn;
        } else {   // held total force of a kinematic particle: f - gamma * (du/dt) (see particle_update)
            const double vkx = __ddiv_rn(P.g.dux[g], P.dt), vky = __ddiv_rn(P.g.duy[g], P.dt), vkz = __ddiv_rn(P.g.duz[g], P.dt);
            fd[p] = make_double4(sub<EXACT>(fx, mul<EXACT>(P.gamma, vkx)), sub<EXACT>(fy, mul<EXACT>(P.gamma, vky)),
                                 sub<EXACT>(fz, mul<EXACT>(P.gamma, vkz)), 0.0);
        }
    }
}

}  // namespace lsmk
