// hydro_impl.cuh -- fused hydrodynamic LB kernel and its launcher, instantiated for one element
// type per translation unit (hydro_f64.cu, hydro_f32.cu define ACM_T and include this file).
#include "kernels.h"
#include "lb_math.cuh"

namespace acm {

// ------------------------------------------------------------------------------------------
// Kernel 2: fused hydrodynamic LB step (Alg. 2; eqs. 8, 10-22, 24, 25, 30)
//   pull g -> p*, j, P -> rho, tau, s_nu, grad/lap of the NEW phi, mu_phi -> F_s+F_p+F_mu+F_b ->
//   u_new = j + F/(2 rho) -> closed-form MRT collision (second-order moments relaxed with s_nu,
//   all others with 1) -> store g (own cell, see header), u_new.
//   g*_i = g^eq_i(u_new) + F_i/2 + (1 - s_nu) 4.5 w_i (e_ia e_ib - d_ab/3) Pi_ab,
//   Pi = P - p*/3 I - u_new u_new^T;  F_mu = -tau s_nu (P - p*/3 I - u_old u_old^T) grad rho
// ------------------------------------------------------------------------------------------
// HVAR = 1: the operator variants of lb_math.cuh (bulk moment relaxed with 1, sub-iterated velocity), switched by a.bulk_one / a.subiter
template <typename T, int Q, bool WALLS, int STATE, bool PEER = false, int HVAR = 0>
__global__ void __launch_bounds__(ACM_MAXT, (WALLS && ACM_HYDRO_MINB > 2) ? 2 : ACM_HYDRO_MINB) hydro_kernel(const HydroArgs<T> a)
{
    int x, y, z;
    if (!cell_of_thread(a.g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(a.g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    const size_t N = a.N;      // zero-extended 32-bit value

    T g[Q];
    load_incoming<Q, T, WALLS, STATE, PEER>(a.Gsrc, N, nb, g, a.Gpeer);
    const T uox = a.U[idx], uoy = a.U[N + idx], uoz = a.U[2 * N + idx];
    const T c0 = __ldg(a.C + idx);
    T gpx, gpy, gpz, lap;
    if constexpr (PEER) fd_phi_peer<Q, T, true>(a.C, nb, a.Cpeer, c0, gpx, gpy, gpz, lap);
    else fd_phi<Q, T, true>(a.C, nb, c0, gpx, gpy, gpz, lap);

    Moments<Q, T, true> m;
    m.compute(g);
    const HydroCell<T> hc = hydro_velocity<T, Q, HVAR>(m, c0, gpx, gpy, gpz, lap, uox, uoy, uoz, a);
    a.U[idx] = hc.ux; a.U[N + idx] = hc.uy; a.U[2 * N + idx] = hc.uz;
    hydro_collide<T, Q, HVAR>(m, hc, a, [&](auto ic, T v) {
        st_stream(outgoing_ptr<Q, decltype(ic)::value, T, WALLS, STATE>(a.Gdst, N, nb), v);
    });
}

template <typename T, int Q, bool WALLS>
static void launch_hydro_state(int state, const Launch& l, const HydroArgs<T>& a)
{
    if (a.Gpeer.lo) {      // peer mode of a slab: two-grid storage only
        hydro_kernel<T, Q, WALLS, ST_POST, true><<<l.grid, l.block, 0, l.stream>>>(a);
        return;
    }
    if (a.bulk_one || a.subiter > 1) {      // operator variants (not available in peer mode: acm.cu rejects the combination)
        if (state == ST_POST) hydro_kernel<T, Q, WALLS, ST_POST, false, 1><<<l.grid, l.block, 0, l.stream>>>(a);
        else if (state == ST_IN) hydro_kernel<T, Q, WALLS, ST_IN, false, 1><<<l.grid, l.block, 0, l.stream>>>(a);
        else hydro_kernel<T, Q, WALLS, ST_SWAP, false, 1><<<l.grid, l.block, 0, l.stream>>>(a);
        return;
    }
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
    if (Q == 9) launch_hydro_q<T, 9>(walls, state, l, a);
    else if (Q == 15) launch_hydro_q<T, 15>(walls, state, l, a);
    else if (Q == 19) launch_hydro_q<T, 19>(walls, state, l, a);
    else launch_hydro_q<T, 27>(walls, state, l, a);
    return cudaGetLastError();
}

template cudaError_t launch_hydro<ACM_T>(int, bool, int, const Launch&, const HydroArgs<ACM_T>&);

}  // namespace acm
