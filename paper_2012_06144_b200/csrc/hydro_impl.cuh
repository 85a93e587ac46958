// hydro_impl.cuh -- fused hydrodynamic LB kernel and its launcher, instantiated for one element
// type per translation unit (hydro_f64.cu, hydro_f32.cu define ACM_T and include this file).
#include "kernels.h"

namespace acm {

// ------------------------------------------------------------------------------------------
// Kernel 2: fused hydrodynamic LB step (Alg. 2; eqs. 8, 10-22, 24, 25, 30)
//   pull g -> p*, j, P -> rho, tau, s_nu, grad/lap of the NEW phi, mu_phi -> F_s+F_p+F_mu+F_b ->
//   u_new = j + F/(2 rho) -> closed-form MRT collision (second-order moments relaxed with s_nu,
//   all others with 1) -> store g (own cell, see header), u_new.
//   g*_i = g^eq_i(u_new) + F_i/2 + (1 - s_nu) 4.5 w_i (e_ia e_ib - d_ab/3) Pi_ab,
//   Pi = P - p*/3 I - u_new u_new^T;  F_mu = -tau s_nu (P - p*/3 I - u_old u_old^T) grad rho
// ------------------------------------------------------------------------------------------
template <typename T, int Q, bool WALLS, int STATE>
__global__ void __launch_bounds__(ACM_MAXT, ACM_HYDRO_MINB) hydro_kernel(const HydroArgs<T> a)
{
    int x, y, z;
    if (!cell_of_thread(a.g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(a.g, x, y, z);
    const int idx = nb.at<0, 0, 0>();
    const size_t N = a.N;

    T g[Q];
    load_incoming<Q, T, WALLS, STATE>(a.Gsrc, N, nb, g);
    const T uox = a.U[idx], uoy = a.U[N + idx], uoz = a.U[2 * N + idx];
    const T c0 = __ldg(a.C + idx);
    T gpx, gpy, gpz, lap;
    fd_phi<Q, T, true>(a.C, nb, c0, gpx, gpy, gpz, lap);

    Moments<Q, T, true> m;
    m.compute(g);
    const T pstar = m.m0;
    const T p3 = pstar * T(1.0 / 3.0);

    const T rho = a.rho_L + c0 * a.drho;                  // eq. 8 (phi_L = 0)
    const T inv_rho = T(1) / rho;
    const T tau = a.tau_L + c0 * a.dtau;                  // eq. 20
    const T s_nu = T(1) / (tau + T(0.5));                 // eq. 21
    const T mu = a.beta4 * c0 * (c0 - T(1)) * (c0 - T(0.5)) - a.kappa * lap;   // eq. 17
    const T grx = a.drho * gpx, gry = a.drho * gpy, grz = a.drho * gpz;

    // deviatoric second moment without the velocity part
    const T Sxx = m.Pxx - p3, Syy = m.Pyy - p3, Szz = m.Pzz - p3;
    // viscous force with the velocity of the previous step (eq. 18)
    const T ts = -tau * s_nu;
    const T oxx = Sxx - uox * uox, oyy = Syy - uoy * uoy, ozz = Szz - uoz * uoz;
    const T oxy = m.Pxy - uox * uoy, oxz = m.Pxz - uox * uoz, oyz = m.Pyz - uoy * uoz;
    const T Fx = mu * gpx - p3 * grx + ts * (oxx * grx + oxy * gry + oxz * grz) + rho * a.gx;
    const T Fy = mu * gpy - p3 * gry + ts * (oxy * grx + oyy * gry + oyz * grz) + rho * a.gy;
    const T Fz = mu * gpz - p3 * grz + ts * (oxz * grx + oyz * gry + ozz * grz) + rho * a.gz;
    // velocity, eq. 22
    const T hx = T(0.5) * Fx * inv_rho, hy = T(0.5) * Fy * inv_rho, hz = T(0.5) * Fz * inv_rho;
    const T ux = m.jx + hx, uy = m.jy + hy, uz = m.jz + hz;
    a.U[idx] = ux; a.U[N + idx] = uy; a.U[2 * N + idx] = uz;

    // collision
    const T om = T(1) - s_nu;
    const T nxx = Sxx - ux * ux, nyy = Syy - uy * uy, nzz = Szz - uz * uz;
    const T k45 = T(4.5) * om, s45 = T(4.5);
    const T Txx = s45 * ux * ux + k45 * nxx, Tyy = s45 * uy * uy + k45 * nyy, Tzz = s45 * uz * uz + k45 * nzz;
    const T Txy = s45 * ux * uy + k45 * (m.Pxy - ux * uy);
    const T Txz = s45 * ux * uz + k45 * (m.Pxz - ux * uz);
    const T Tyz = s45 * uy * uz + k45 * (m.Pyz - uy * uz);
    const T A = pstar - T(1.5) * (ux * ux + uy * uy + uz * uz) - T(1.5) * om * (nxx + nyy + nzz);
    const T bx = T(3) * (ux + hx), by = T(3) * (uy + hy), bz = T(3) * (uz + hz);
    emit_populations<Q, T>(A, bx, by, bz, Txx, Tyy, Tzz, Txy, Txz, Tyz, [&](auto ic, T v) {
        st_stream(outgoing_ptr<Q, decltype(ic)::value, T, WALLS, STATE>(a.Gdst, N, nb), v);
    });
}

template <typename T, int Q, bool WALLS>
static void launch_hydro_state(int state, const Launch& l, const HydroArgs<T>& a)
{
    if (state == ST_POST) hydro_kernel<T, Q, WALLS, ST_POST><<<l.grid, l.block, 0, l.stream>>>(a);
    else if (state == ST_IN) hydro_kernel<T, Q, WALLS, ST_IN><<<l.grid, l.block, 0, l.stream>>>(a);
    else hydro_kernel<T, Q, WALLS, ST_SWAP><<<l.grid, l.block, 0, l.stream>>>(a);
}

template <typename T, int Q>
static void launch_hydro_q(bool walls, int state, const Launch& l, const HydroArgs<T>& a)
{
    if (walls) launch_hydro_state<T, Q, true>(state, l, a);
    else launch_hydro_state<T, Q, false>(state, l, a);
}

template <typename T>
cudaError_t launch_hydro(int Q, bool walls, int state, const Launch& l, const HydroArgs<T>& a)
{
    if (Q == 15) launch_hydro_q<T, 15>(walls, state, l, a);
    else if (Q == 19) launch_hydro_q<T, 19>(walls, state, l, a);
    else launch_hydro_q<T, 27>(walls, state, l, a);
    return cudaGetLastError();
}

template cudaError_t launch_hydro<ACM_T>(int, bool, int, const Launch&, const HydroArgs<ACM_T>&);

}  // namespace acm
