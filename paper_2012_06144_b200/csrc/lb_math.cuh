// lb_math.cuh -- the per-cell arithmetic of the two LB steps as device functions, shared by the fused
// kernels (phase_impl.cuh, hydro_impl.cuh: Algorithm 2) and the unfused six-kernel pipeline
// (unfused_impl.cuh: Algorithm 1), so that both evaluate exactly the same expressions.
#pragma once
#include "common.cuh"
#include "vec2.cuh"

namespace acm {

// Phase-field collision at one cell (eqs. 4-6): from the streamed populations h (their
// moments m, phi = m.m0), the OLD phi at the cell (c0) and its gradient (gx,gy,gz), and u, emit the
// post-collision populations through store(ic, value).
template <typename T, int Q, int COLL, typename Store>
__device__ __forceinline__ void phase_collide(const T (&h)[Q], const Moments<Q, T, false>& m, T c0, T gx, T gy, T gz, T ux, T uy,
                                              T uz, T one_minus_omega, T inv_xi, T ref, Store&& store)
{
    // fp32 instance (A22): h and phi are stored as deviations from the reference phase `ref` (0 or 1),
    // h_i - ref w_i and phi - ref, so that the bulk of that phase keeps its digits; fp64: ref = 0, nothing changes
    constexpr bool DEV = is_f32<T>;
    const T phid = m.m0;                             // stored zeroth moment
    const T phi = DEV ? ref + phid : phid;           // the order parameter itself
    // interface normal (n = 0 where grad phi vanishes exactly) and theta = (1 - 4 (phi-1/2)^2)/xi
    const T g2 = gx * gx + gy * gy + gz * gz;
    const T inv = inv_norm_or_zero(g2);
    T theta;
    if constexpr (DEV) {
        theta = T(4) * (ref + c0) * ((T(1) - ref) - c0) * inv_xi;     // 1 - 4 (phi - 1/2)^2 = 4 phi (1 - phi), c0 = phi_old - ref
    } else {
        const T dc = c0 - T(0.5);
        theta = (T(1) - T(4) * dc * dc) * inv_xi;
    }
    const T tnx = theta * inv * gx, tny = theta * inv * gy, tnz = theta * inv * gz;   // theta * n

    // closed form of the collision: h*_i = w_i [A + e_i.b + e_i e_i : T] (+ keep * h_i for SRT)
    T A, bx, by, bz, Ts, keep;
    if constexpr (COLL == PHASE_MRT) {
        // first-order moments relaxed with omega_phi, all others with 1 (A3):
        // with d = j - phi u + (theta/6) n:  h*_i = phi Gamma_i(u) + F_i/2 + (1-omega) 3 w_i e_i.d
        const T k = T(3) * one_minus_omega;
        const T sixth = T(1.0 / 6.0);
        const T dxm = m.jx - phi * ux + sixth * tnx;
        const T dym = m.jy - phi * uy + sixth * tny;
        const T dzm = m.jz - phi * uz + sixth * tnz;
        const T p3 = T(3) * phi;
        const T usq = T(1.5) * (ux * ux + uy * uy + uz * uz);
        A = DEV ? phid * (T(1) - usq) - ref * usq : phi * (T(1) - usq);        // DEV: phi (1 - usq) - ref
        bx = p3 * ux + T(0.5) * tnx + k * dxm;
        by = p3 * uy + T(0.5) * tny + k * dym;
        bz = p3 * uz + T(0.5) * tnz + k * dzm;
        Ts = T(4.5) * phi;
        keep = T(0);
    } else {
        // single relaxation time (A23): h*_i = (1-omega) h_i + omega phi Gamma_i(u) + (1-omega/2) F_i
        const T omega = T(1) - one_minus_omega;
        const T op = omega * phi, fh = T(1) - T(0.5) * omega;
        const T usq = T(1.5) * (ux * ux + uy * uy + uz * uz);
        // DEV: (1-omega) ref w_i + omega phi w_i (1 - usq) - ref w_i = w_i omega [phid (1 - usq) - ref usq]
        A = DEV ? omega * (phid * (T(1) - usq) - ref * usq) : op * (T(1) - usq);
        bx = T(3) * op * ux + fh * tnx;
        by = T(3) * op * uy + fh * tny;
        bz = T(3) * op * uz + fh * tnz;
        Ts = T(4.5) * op;
        keep = one_minus_omega;
    }
    auto post = [&](auto ic, T v) -> T {
        if constexpr (COLL == PHASE_SRT) return v + keep * h[decltype(ic)::value];
        else return v;
    };
    if constexpr (!DEV) {
        emit_populations<Q, T>(A, bx, by, bz, Ts * ux * ux, Ts * uy * uy, Ts * uz * uz, Ts * ux * uy, Ts * ux * uz,
                               Ts * uy * uz, [&](auto ic, T v) {
                                   store(ic, post(ic, v));
                               });
    } else {
        // fp32 instance (reading A22): the rest population is set by subtraction,
        // h*_0 = phi_new - sum_{i>=1} h*_i, so that the collision conserves phi exactly in fp32
        // (all of them as deviations from ref w_i, which sum to ref).
        T rest = phid;
        emit_populations<Q, T>(A, bx, by, bz, Ts * ux * ux, Ts * uy * uy, Ts * uz * uz, Ts * ux * uy, Ts * ux * uz,
                               Ts * uy * uz, [&](auto ic, T v) {
                                   constexpr int i = decltype(ic)::value;
                                   if constexpr (i > 0) {
                                       const T o = post(ic, v);
                                       rest -= o;
                                       store(ic, o);
                                   }
                               });
        store(std::integral_constant<int, 0>{}, rest);
    }
}

// Hydrodynamic forces and velocity at one cell (eqs. 8, 13-22, 30): from the moments m of the incoming
// populations g, the NEW phi at the cell (c0) with its gradient and Laplacian, and the velocity of the
// previous step (uo), compute u_new = j + F/(2 rho) and keep what the collision needs.
template <typename T>
struct HydroCell {
    T ux, uy, uz;      // u_new, eq. 22
    T hx, hy, hz;      // F/(2 rho)
    T s_nu;            // eq. 21
    T Sxx, Syy, Szz;   // P_aa - p*/3
};

// HVAR = 0: the default operators (readings A4, A10).  HVAR = 1: the variants of SURVEY 8(f)-2 switched by the
// run-time fields of HydroArgs -- a.bulk_one (A26: the bulk moment relaxes with 1, only the deviatoric second-order
// moments with s_nu) and a.subiter (A27: that many sweeps of the fixed point of eq. 22).
// T is the element type the arithmetic runs in (a cell, or a pair of cells: vec2.cuh), S the scalar type of the arguments.
template <typename T, int Q, int HVAR = 0, typename S>
__device__ __forceinline__ HydroCell<T> hydro_velocity(const Moments<Q, T, true>& m, T c0, T gpx, T gpy, T gpz, T lap, T uox, T uoy,
                                                       T uoz, const HydroArgs<S>& a)
{
    const T pstar = m.m0;
    const T p3 = pstar * T(1.0 / 3.0);

    // fp32 instance: c0 = phi - ref (see phase_collide); a.rho_L and a.tau_L then hold the values AT phi = ref
    const T rho = a.rho_L + c0 * a.drho;                  // eq. 8 (phi_L = 0)
    const T inv_rho = T(1) / rho;
    const T tau = a.tau_L + c0 * a.dtau;                  // eq. 20
    const T s_nu = T(1) / (tau + T(0.5));                 // eq. 21
    T mu;                                                 // eq. 17
    if constexpr (is_f32<T>) mu = a.beta4 * (a.ref + c0) * (c0 - (T(1) - a.ref)) * (c0 + (a.ref - T(0.5))) - a.kappa * lap;
    else mu = a.beta4 * c0 * (c0 - T(1)) * (c0 - T(0.5)) - a.kappa * lap;
    const T grx = a.drho * gpx, gry = a.drho * gpy, grz = a.drho * gpz;

    // deviatoric second moment without the velocity part
    const T Sxx = m.Pxx - p3, Syy = m.Pyy - p3, Szz = m.Pzz - p3;
    // the parts of F that do not depend on u: F_s + F_p (eqs. 14, 16) and F_b (eq. 30)
    const T F0x = mu * gpx - p3 * grx, F0y = mu * gpy - p3 * gry, F0z = mu * gpz - p3 * grz;
    const T Fbx = rho * a.gx, Fby = rho * a.gy, Fbz = rho * a.gz;
    const T ts = -tau * s_nu;
    T hx, hy, hz, ux, uy, uz;
    const int sweeps = HVAR ? a.subiter : 1;
    for (int sweep = 0; sweep < sweeps; ++sweep) {
        // viscous force (eq. 18) with the velocity of the previous step, or of the previous sweep
        const T oxx = Sxx - uox * uox, oyy = Syy - uoy * uoy, ozz = Szz - uoz * uoz;
        const T oxy = m.Pxy - uox * uoy, oxz = m.Pxz - uox * uoz, oyz = m.Pyz - uoy * uoz;
        T Fx = F0x + ts * (oxx * grx + oxy * gry + oxz * grz) + Fbx;
        T Fy = F0y + ts * (oxy * grx + oyy * gry + oyz * grz) + Fby;
        T Fz = F0z + ts * (oxz * grx + oyz * gry + ozz * grz) + Fbz;
        if constexpr (HVAR != 0) {
            if (a.bulk_one) {
                // second moment of Omega (g - g^eq) = s_nu Pi_dev + (tr Pi / D) I  instead of s_nu Pi
                const T tr = Lat<Q>::DIM == 3 ? oxx + oyy + ozz : oxx + oyy;
                const T tb = -tau * (T(1) - s_nu) * tr * T(1.0 / Lat<Q>::DIM);
                Fx += tb * grx; Fy += tb * gry; Fz += tb * grz;
            }
        }
        // velocity, eq. 22
        hx = T(0.5) * Fx * inv_rho; hy = T(0.5) * Fy * inv_rho; hz = T(0.5) * Fz * inv_rho;
        ux = m.jx + hx; uy = m.jy + hy; uz = m.jz + hz;
        uox = ux; uoy = uy; uoz = uz;
    }
    return HydroCell<T>{ux, uy, uz, hx, hy, hz, s_nu, Sxx, Syy, Szz};
}

// Coefficients of a closed-form collision result  f*_i = w_i [A + e_i.b + e_i e_i : T]  (T symmetric).  Because all
// moments beyond the first (phase field) / second (hydrodynamics) order relax with rate 1, these ten numbers ARE the
// post-collision state of a cell: the moment representation of moment_impl.cuh stores them instead of the populations.
template <typename T>
struct Coeffs {
    T A, bx, by, bz, Txx, Tyy, Tzz, Txy, Txz, Tyz;
};

// Hydrodynamic collision at one cell (eqs. 10-12, 25 in closed form): the coefficients of g*.
template <typename T, int Q, int HVAR = 0, typename S>
__device__ __forceinline__ Coeffs<T> hydro_coeffs(const Moments<Q, T, true>& m, const HydroCell<T>& hc, const HydroArgs<S>& a)
{
    const T pstar = m.m0;
    const T ux = hc.ux, uy = hc.uy, uz = hc.uz, hx = hc.hx, hy = hc.hy, hz = hc.hz, s_nu = hc.s_nu;
    const T Sxx = hc.Sxx, Syy = hc.Syy, Szz = hc.Szz;
    // collision
    const T om = T(1) - s_nu;
    const T nxx = Sxx - ux * ux, nyy = Syy - uy * uy, nzz = Szz - uz * uz;
    const T k45 = T(4.5) * om, s45 = T(4.5);
    T Txx = s45 * ux * ux + k45 * nxx, Tyy = s45 * uy * uy + k45 * nyy, Tzz = s45 * uz * uz + k45 * nzz;
    const T Txy = s45 * ux * uy + k45 * (m.Pxy - ux * uy);
    const T Txz = s45 * ux * uz + k45 * (m.Pxz - ux * uz);
    const T Tyz = s45 * uy * uz + k45 * (m.Pyz - uy * uz);
    // trace of Pi over the lattice's dimensions (D2Q9: the plane only; u_z = 0 there)
    const T trPi = Lat<Q>::DIM == 3 ? nxx + nyy + nzz : nxx + nyy;
    T A = pstar - T(1.5) * (ux * ux + uy * uy + uz * uz) - T(1.5) * om * trPi;
    if constexpr (HVAR != 0) {
        if (a.bulk_one) {
            // Omega^g = I - (1 - s_nu)(P_2 - P_trace), P_trace x = w_i (|e_i|^2 - D/3) tr Pi(x) / (sum w t^2): Pi becomes trace-free
            constexpr double inv_norm = Lat<Q>::DIM == 3 ? 1.5 : 2.25;       // 1 / sum_i w_i (|e_i|^2 - D/3)^2
            const T t = T(inv_norm) * om * trPi;
            Txx -= t; Tyy -= t; Tzz -= t;
            A += T(1.5) * om * trPi;
        }
    }
    const T bx = T(3) * (ux + hx), by = T(3) * (uy + hy), bz = T(3) * (uz + hz);
    return Coeffs<T>{A, bx, by, bz, Txx, Tyy, Tzz, Txy, Txz, Tyz};
}

// ... and the populations they stand for, emitted through store(ic, value).
template <typename T, int Q, int HVAR = 0, typename S, typename Store>
__device__ __forceinline__ void hydro_collide(const Moments<Q, T, true>& m, const HydroCell<T>& hc, const HydroArgs<S>& a, Store&& store)
{
    const Coeffs<T> k = hydro_coeffs<T, Q, HVAR>(m, hc, a);
    emit_populations<Q, T>(k.A, k.bx, k.by, k.bz, k.Txx, k.Tyy, k.Tzz, k.Txy, k.Txz, k.Tyz, store);
}

}  // namespace acm
