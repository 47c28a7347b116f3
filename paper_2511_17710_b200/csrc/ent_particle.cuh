// ent_particle.cuh -- one particle through sub-steps 3-8.  Used by the untiled and the tiled kernels.
#pragma once
#include "ent_dev.cuh"

namespace ent {

// ---------------------------------------------------------------------------------------------------------
// S1-S5 for one particle.  In: cell indices i[], offsets d[], phi, u[].  Out: the same, advanced by one step;
// di[] = un-wrapped cell shift per dimension (for the deposit), alive = false if it left through an ABSORB side.
// eps = (q/m) dt / 2.
// ---------------------------------------------------------------------------------------------------------
// push_from_fields: everything after the gather (EB = the six interpolated contravariant components).
struct NoGeo {};                          // Cartesian grids need no node factors

// The divisions of the fp32 displacement form are MUFU.RCP quotients (__fdividef, 2 ulp): increments of at most one cell, so 2.4e-7
// cells at worst against the 1e-5 bar.
// atan2(y, x) and log1p(x) with a short series where the argument is small (the displacement of one step is a small fraction
// of r), the library routine otherwise; truncation error below 2e-12
// sqrt.approx.f32 (MUFU.SQRT, relative error 2^-23, exact zero for zero) instead of the IEEE sequence
__device__ __forceinline__ float sqrt_approx(float x) { float r; asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float atan2_step(float y, float x) {
    if (x > 0.f && fabsf(y) < 0.0625f * x) {
        const float t = __fdividef(y, x), t2 = t * t;
        return t * fmaf(t2, fmaf(t2, fmaf(t2, -1.0f / 7.0f, 0.2f), -1.0f / 3.0f), 1.0f);
    }
    return atan2f(y, x);
}
__device__ __forceinline__ float log1p_step(float x) {
    if (fabsf(x) < 0.015f) return x * fmaf(x, fmaf(x, fmaf(x, fmaf(x, 0.2f, -0.25f), 1.0f / 3.0f), -0.5f), 1.0f);
    return log1pf(x);
}
template <int D, int KIND, class GEO>
__device__ __forceinline__ void push_from_fields_geo(const GridDev &g, const GEO &geo, const float EB[6], int i[3], float d[3], float &phi,
                                                     float u[3], float eps, float dt, int di[3], bool &alive) {
    float E[3], B[3];
    if (KIND == ENT_CART) {
        // step 4: A^hat = sqrt(h_ii) A^i; Cartesian code basis is already aligned with x,y,z
#pragma unroll
        for (int a = 0; a < 3; ++a) { E[a] = g.dx[a] * EB[a]; B[a] = g.dx[a] * EB[3 + a]; }
        push_momentum(g, u, E, B, eps);                                                  // step 5, Eq. 3
        float ig = inv_gamma(u);
#pragma unroll
        for (int a = 0; a < 3; ++a) {                                         // steps 6-7
            if (a < D) {
                float x = d[a] + (u[a] * ig) * (dt * g.inv_dx[a]);
                split_offset(x, di[a], d[a]);
            } else di[a] = 0;
        }
    } else if (!g.curv_f64) {
        // axisymmetric, fp32 DISPLACEMENT form: the step v dt is projected on the local frame
        // (r, theta, phi)-hat at the old point and turned into increments of the code coordinates, which are added to the in-cell
        // offsets exactly as on the Cartesian grids; no absolute position is ever formed in fp32.  Same mathematics as the
        // global-Cartesian round trip of P:147-153, P:285-327 (the oracle's), which in fp32 would lose the displacement.
        SphF s{};
        if constexpr (KIND != ENT_CART) s = sphf_of_code<KIND>(g, geo, i[0], d[0], i[1], d[1]);
        float sp, cp;
        sincos_azimuth(phi, sp, cp);
        {   // step 4: tetrad (at the particle, G2) then rotation (r,th,phi)-hat -> (x,y,z)-hat
            float Ar = s.sh1 * EB[0], At = s.sh2 * EB[1], Ap = s.sh3 * EB[2];
            E[0] = Ar * s.st * cp + At * s.ct * cp - Ap * sp;
            E[1] = Ar * s.st * sp + At * s.ct * sp + Ap * cp;
            E[2] = Ar * s.ct - At * s.st;
            Ar = s.sh1 * EB[3]; At = s.sh2 * EB[4]; Ap = s.sh3 * EB[5];
            B[0] = Ar * s.st * cp + At * s.ct * cp - Ap * sp;
            B[1] = Ar * s.st * sp + At * s.ct * sp + Ap * cp;
            B[2] = Ar * s.ct - At * s.st;
        }
        push_momentum(g, u, E, B, eps);
        const float ig = inv_gamma(u);
        const float Dx = (u[0] * ig) * dt, Dy = (u[1] * ig) * dt, Dz = (u[2] * ig) * dt;
        const float Dh = Dx * cp + Dy * sp;                                   // component along the old cylindrical radius
        const float dr_ = Dh * s.st + Dz * s.ct, dth_ = Dh * s.ct - Dz * s.st, dph_ = Dy * cp - Dx * sp;
        const float rp = s.r + dr_;
        const float d2 = dr_ * dr_ + dth_ * dth_ + dph_ * dph_;
        const float rn = sqrt_approx(rp * rp + dth_ * dth_ + dph_ * dph_);
        const float Dr = __fdividef(2.0f * s.r * dr_ + d2, rn + s.r);                 // r' - r without cancellation
        const float a = rp * s.st + dth_ * s.ct;                               // new cylindrical radius vector in the old meridional plane
        const float rho = sqrt_approx(a * a + dph_ * dph_);
        const float zn = rp * s.ct - dth_ * s.st;
        const float rma = a > 0.f ? __fdividef(dph_ * dph_, rho + a) : rho - a;       // rho' - a
        const float Dth = atan2_step(dth_ + rma * s.ct, zn * s.ct + rho * s.st);   // theta' - theta
        const float Dph = atan2_step(dph_, a);
        float x1n, x2n;
        if (KIND == ENT_SPH) { x1n = __fdividef(Dr, g.drf); x2n = __fdividef(Dth, g.dthf); }
        else {
            x1n = __fdividef(log1p_step(__fdividef(Dr, s.rr0)), g.dRf);
            float DT = Dth;
            if (g.vtf != 0.f) {                                               // theta(T + DT) - theta(T) = Dth: theta is a cubic, so its
                const float c3 = 4.0f * g.vtf * 0.101321183642337771f;        // Taylor series ends: th1 DT + c2 DT^2 + c3 DT^3, c3 = 4 vt / pi^2
                DT = __fdividef(Dth, s.th1);
#pragma unroll
                for (int it = 0; it < 2; ++it) {                              // two Newton steps from the linear guess (no cube root, cf. App. B)
                    const float f = ((c3 * DT + s.c2) * DT + s.th1) * DT - Dth;
                    const float fp = (3.0f * c3 * DT + 2.0f * s.c2) * DT + s.th1;
                    DT -= __fdividef(f, fp);
                }
            }
            x2n = __fdividef(DT, g.dTf);
        }
        split_offset(d[0] + x1n, di[0], d[0]);
        split_offset(d[1] + x2n, di[1], d[1]);
        di[2] = 0;
        float phn = phi + Dph;
        // wrap into [0, 2 pi) with the two-constant form 2 pi = TWO_PI_F - TWO_PI_LO (TWO_PI_F alone is 1.75e-7 above 2 pi, which is
        // most of an fp32 ulp of an azimuth near 2 pi and showed up in the full-size parity of C5)
        if (phn >= TWO_PI_F) phn = (phn - TWO_PI_F) + TWO_PI_LO;
        if (phn < 0.f) phn = (phn - TWO_PI_LO) + TWO_PI_F;
        if (phn >= TWO_PI_F) phn = 0.f;
        phi = phn;
    } else {
        // axisymmetric, fp64 maps through the global Cartesian frame (ENT_OPT_CURV_FP64 = 1; the round-1 form, kept for A/B)
        // particle at (x1, x2, phi)
        double x1 = (double)i[0] + (double)d[0], x2 = (double)i[1] + (double)d[1], ph = (double)phi;
        Sph s = sph_of_code<KIND>(g, x1, x2);
        double st, ct, sp, cp;
        sincos(s.th, &st, &ct);
        sincos(ph, &sp, &cp);
        {   // step 4: tetrad (at the particle, G2) then rotation (r,th,phi)-hat -> (x,y,z)-hat
            float fst = (float)st, fct = (float)ct, fsp = (float)sp, fcp = (float)cp;
            float h1 = (float)s.sh1, h2 = (float)s.sh2, h3 = (float)s.sh3;
            float Ar = h1 * EB[0], At = h2 * EB[1], Ap = h3 * EB[2];
            E[0] = Ar * fst * fcp + At * fct * fcp - Ap * fsp;
            E[1] = Ar * fst * fsp + At * fct * fsp + Ap * fcp;
            E[2] = Ar * fct - At * fst;
            Ar = h1 * EB[3]; At = h2 * EB[4]; Ap = h3 * EB[5];
            B[0] = Ar * fst * fcp + At * fct * fcp - Ap * fsp;
            B[1] = Ar * fst * fsp + At * fct * fsp + Ap * fcp;
            B[2] = Ar * fct - At * fst;
        }
        push_momentum(g, u, E, B, eps);
        float ig = inv_gamma(u);
        // step 6: x^X += u/gamma dt in the global Cartesian frame
        double X = s.r * st * cp + (double)(u[0] * ig) * (double)dt;
        double Y = s.r * st * sp + (double)(u[1] * ig) * (double)dt;
        double Z = s.r * ct + (double)(u[2] * ig) * (double)dt;
        // step 7: back to code coordinates
        double rho2 = X * X + Y * Y;
        double rn = sqrt(rho2 + Z * Z);
        double thn = 0.5 * PI_D - atan2(Z, sqrt(rho2));
        double phn = PI_D - atan2(Y, -X);
        double y1, y2;
        if (KIND == ENT_SPH) { y1 = (rn - g.rmin) / g.dr; y2 = thn / g.dth; }
        else { y1 = (log(rn - g.r0) - g.Rmin) / g.dR; double T_old = x2 * g.dT; y2 = T_of_theta(g.vt, thn, T_old + (thn - s.th) / dtheta_dT(g.vt, T_old)) / g.dT; }
        float phf = (float)phn;
        if (phf >= TWO_PI_F) phf -= TWO_PI_F;
        if (phf < 0.f) phf = 0.f;
        phi = phf;
        double f1 = floor(y1), f2 = floor(y2);
        int n1 = (int)f1, n2 = (int)f2;
        float e1 = (float)(y1 - f1), e2 = (float)(y2 - f2);
        if (e1 >= 1.0f) { e1 = 0.f; n1 += 1; }                                // rounding to fp32 reached the upper face
        if (e2 >= 1.0f) { e2 = 0.f; n2 += 1; }
        di[0] = n1 - i[0]; di[1] = n2 - i[1]; di[2] = 0;
        d[0] = e1; d[1] = e2;
    }
    // O7 crossing bookkeeping
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (a >= D) continue;
        int in = i[a] + di[a];
        if (g.bc[a] == ENT_PERIODIC) {
            if (in < 0) in += g.N[a];
            if (in >= g.N[a]) in -= g.N[a];
        } else if (g.bc[a] == ENT_AXIS) {
            if (in >= g.N[a]) { in = g.N[a] - 1; d[a] = 0.99999994f; di[a] = in - i[a]; }   // theta = pi exactly (G11)
            if (in < 0) { in = 0; d[a] = 0.f; di[a] = in - i[a]; }
        } else {                                                              // ABSORB (G9)
            if (in < 0) { alive = false; in = 0; }
            if (in >= g.N[a]) { alive = false; in = g.N[a] - 1; }
        }
        i[a] = in;
    }
}

template <int D, int KIND>
__device__ __forceinline__ void push_from_fields(const GridDev &g, const float EB[6], int i[3], float d[3], float &phi,
                                                 float u[3], float eps, float dt, int di[3], bool &alive) {
    if constexpr (KIND == ENT_CART) push_from_fields_geo<D, KIND>(g, NoGeo{}, EB, i, d, phi, u, eps, dt, di, alive);
    else push_from_fields_geo<D, KIND>(g, GlobalGeo<KIND>{g}, EB, i, d, phi, u, eps, dt, di, alive);
}

template <int D, int KIND, class Loader>
__device__ __forceinline__ void push_particle(const GridDev &g, const Loader &ld, int i[3], float d[3], float &phi,
                                              float u[3], float eps, float dt, int di[3], bool &alive) {
    float EB[6];
    gather<D>(g, ld, i, d, EB);                                               // step 3
    push_from_fields<D, KIND>(g, EB, i, d, phi, u, eps, dt, di, alive);
}

// ---------------------------------------------------------------------------------------------------------
// S7 deposit for one particle (Eq. 6, step 8 P:155-157, "modified zig-zag" P:575).
// i0[], a[] = old cell and offset; di[] = un-wrapped cell shift in {-1,0,1}; dn[] = new offset;
// Q = q w / dt; qw = q w.  Acc::add(comp, padded_index, value) accumulates one contribution.
// All arithmetic is in the old cell's frame (small numbers only: "(real)(i+delta) is never necessary").
// ---------------------------------------------------------------------------------------------------------
// fp32 add to GLOBAL memory without a return value.  The pointers come out of structs handed to out-of-line functions, where the
// compiler no longer knows their state space and would emit the generic atomic (with its shared-memory compare-and-swap branch).
__device__ __forceinline__ void red_global_f32(float *p, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(__cvta_generic_to_global(p)), "f"(v) : "memory");
}
struct GlobalAcc {
    float *const *J;
    __device__ __forceinline__ void add(int comp, long long idx, float v) const { red_global_f32(J[comp] + idx, v); }
    // four contributions at once (an accumulator may treat them together: the shared-memory tile tests their carries with one branch)
    __device__ __forceinline__ void add4(int c0, long long i0, float v0, int c1, long long i1, float v1,
                                         int c2, long long i2, float v2, int c3, long long i3, float v3) const {
        add(c0, i0, v0); add(c1, i1, v1); add(c2, i2, v2); add(c3, i3, v3);
    }
};

template <int D, class Acc>
__device__ __forceinline__ void deposit_segment(const Acc &acc, long long base, long long s1, long long s2,
                                                const float Dv[3], const float W[3], float Q, float hv) {
    if (D == 3) {
        // J^comp at the 4 transverse nodes: Q D_comp [ w(W_a,s_a) w(W_b,s_b) +- D_a D_b / 12 ]  (reading G7)
        const long long st[3] = { 1, s1, s2 };
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            const int a = (comp + 1) % 3, b = (comp + 2) % 3;
            float c = Dv[a] * Dv[b] * (1.0f / 12.0f);
            float QD = Q * Dv[comp];
            float w11 = W[a] * W[b] + c;
            float w10 = W[a] - w11;           // W_a (1 - W_b) - c
            float w01 = W[b] - w11;           // (1 - W_a) W_b - c
            float w00 = 1.0f - W[a] - w01;    // (1 - W_a)(1 - W_b) + c
            acc.add(comp, base, QD * w00);
            acc.add(comp, base + st[a], QD * w10);
            acc.add(comp, base + st[b], QD * w01);
            acc.add(comp, base + st[a] + st[b], QD * w11);
        }
    } else {
        float q0 = Q * Dv[0], q1 = Q * Dv[1];
        acc.add4(0, base, q0 * (1.0f - W[1]), 0, base + s1, q0 * W[1], 1, base, q1 * (1.0f - W[0]), 1, base + 1, q1 * W[0]);
        float h1 = hv * W[1], h0 = hv - h1;                                   // out-of-plane, velocity form (G8)
        acc.add4(2, base, h0 * (1.0f - W[0]), 2, base + 1, h0 * W[0], 2, base + s1, h1 * (1.0f - W[0]), 2, base + s1 + 1, h1 * W[0]);
    }
}

// out-of-plane rate q w v^3_code / 2 per segment for the 2D grids (G8); u = momentum at n+1/2
template <int KIND, class GEO>
__device__ __forceinline__ float half_qw_v3(const GridDev &g, const GEO &geo, const int i0[3], const float a[3], const float b[3],
                                            float phi0, float phi1, const float u[3], float qw) {
    float ig = inv_gamma(u);
    if (KIND == ENT_CART) return 0.5f * qw * (u[2] * ig);                     // h33 = 1
    if (!g.curv_f64) {
        float dphi = phi1 - phi0;                                             // shorter arc
        if (dphi > 3.14159265358979f) dphi -= TWO_PI_F;
        if (dphi <= -3.14159265358979f) dphi += TWO_PI_F;
        SphF s{};
        if constexpr (KIND != ENT_CART) s = sphf_of_code<KIND>(g, geo, i0[0], 0.5f * (a[0] + b[0]), i0[1], 0.5f * (a[1] + b[1]));
        if (s.sh3 < 1e-12f) return 0.f;
        float sp, cp;
        sincos_azimuth(phi0 + 0.5f * dphi, sp, cp);
        return 0.5f * qw * __fdividef((u[1] * cp - u[0] * sp) * ig, s.sh3);
    }
    double dphi = (double)phi1 - (double)phi0;
    dphi -= 2.0 * PI_D * floor((dphi + PI_D) / (2.0 * PI_D));                 // shorter arc
    double phm = (double)phi0 + 0.5 * dphi;
    double x1 = (double)i0[0] + 0.5 * ((double)a[0] + (double)b[0]);
    double x2 = (double)i0[1] + 0.5 * ((double)a[1] + (double)b[1]);
    Sph s = sph_of_code<KIND>(g, x1, x2);
    if (s.sh3 < 1e-12) return 0.f;
    double sp, cp;
    sincos(phm, &sp, &cp);
    double v3 = ((-(double)u[0] * sp + (double)u[1] * cp) * (double)ig) / s.sh3;
    return (float)(0.5 * (double)qw * v3);
}

// gi / ii: the array the contributions are indexed in and the old cell's index in it (the padded global arrays and i0
// itself for the global path; a shared-memory J tile and the cell's box coordinates for the tiled path).
template <int D, int KIND, class Acc, class GEO>
__device__ __forceinline__ void deposit_particle_at(const GridDev &g, const GEO &geo, const Acc &acc, const int i0[3], const float a[3],
                                                    const int di[3], const float dn[3], float phi0, float phi1,
                                                    const float u[3], float qw, float inv_dt, const GridDev &gi, const int ii[3]) {
    float D1[3], W1[3], D2[3], W2[3], b[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        if (k < D) {
            const float fdi = (float)di[k];
            b[k] = fdi + dn[k];                                               // new position in the old cell's frame
            float r = fminf(fminf(fdi, 0.f) + 1.0f, fmaxf(fmaxf(fdi, 0.f), 0.5f * (a[k] + b[k])));   // relay point, branch-free
            D1[k] = r - a[k];  W1[k] = 0.5f * (a[k] + r);
            D2[k] = b[k] - r;  W2[k] = 0.5f * (r + b[k]) - fdi;
        } else { b[k] = 0.f; D1[k] = W1[k] = D2[k] = W2[k] = 0.f; }
    }
    const long long s1 = gi.P[0], s2 = (long long)gi.P[0] * gi.P[1];
    long long base1 = pidx<D>(gi, ii[0], ii[1], ii[2]);
    long long base2 = base1 + di[0] + s1 * di[1] + (D == 3 ? s2 * di[2] : 0);   // un-wrapped: may point into the ghosts
    float Q = qw * inv_dt;
    float hv = 0.f;
    if (D == 2) hv = half_qw_v3<KIND>(g, geo, i0, a, b, phi0, phi1, u, qw);
    deposit_segment<D>(acc, base1, s1, s2, D1, W1, Q, hv);
    deposit_segment<D>(acc, base2, s1, s2, D2, W2, Q, hv);
}

template <int D, int KIND, class Acc>
__device__ __forceinline__ void deposit_particle(const GridDev &g, const Acc &acc, const int i0[3], const float a[3],
                                                 const int di[3], const float dn[3], float phi0, float phi1,
                                                 const float u[3], float qw, float inv_dt) {
    if constexpr (KIND == ENT_CART) deposit_particle_at<D, KIND>(g, NoGeo{}, acc, i0, a, di, dn, phi0, phi1, u, qw, inv_dt, g, i0);
    else deposit_particle_at<D, KIND>(g, GlobalGeo<KIND>{g}, acc, i0, a, di, dn, phi0, phi1, u, qw, inv_dt, g, i0);
}

}  // namespace ent
