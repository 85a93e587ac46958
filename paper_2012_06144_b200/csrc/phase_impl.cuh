// phase_impl.cuh -- fused phase-field LB kernel and its launcher, instantiated for one element
// type per translation unit (phase_f64.cu, phase_f32.cu define ACM_T and include this file).
#include "kernels.h"
#include "lb_math.cuh"

namespace acm {

// ------------------------------------------------------------------------------------------
// Kernel 1: fused phase-field LB step (Alg. 2; eqs. 4-7, 23)
//   pull h -> phi_new = sum h -> grad/normal/theta from the OLD phi -> closed-form MRT collision
//   (first-order moments relaxed with omega_phi, all others with 1) -> store h, phi_new.
// With d = j - phi_new u + (theta/6) n:   h*_i = h^eq_i + F_i/2 + (1-omega_phi) 3 w_i e_i.d
// ------------------------------------------------------------------------------------------
template <typename T, int Q, bool WALLS, int STATE, int COLL, bool PEER = false>
__global__ void __launch_bounds__(ACM_MAXT, (WALLS && ACM_PHASE_MINB > 2) ? 2 : ACM_PHASE_MINB) phase_kernel(const PhaseArgs<T> a)
{
    int x, y, z;
    if (!cell_of_thread(a.g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(a.g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    const size_t N = a.N;      // zero-extended 32-bit value

    T h[Q];
    load_incoming<Q, T, WALLS, STATE, PEER>(a.Hsrc, N, nb, h, a.Hpeer);
    const T ux = __ldg(a.U + idx), uy = __ldg(a.U + N + idx), uz = __ldg(a.U + 2 * N + idx);
    const T c0 = __ldg(a.Csrc + idx);
    T gx, gy, gz, lap_unused;
    if constexpr (PEER) fd_phi_peer<Q, T, false>(a.Csrc, nb, a.Cpeer, c0, gx, gy, gz, lap_unused);
    else fd_phi<Q, T, false>(a.Csrc, nb, c0, gx, gy, gz, lap_unused);

    Moments<Q, T, false> m;
    m.compute(h);
    const T phi = m.m0;

    phase_collide<T, Q, COLL>(h, m, c0, gx, gy, gz, ux, uy, uz, a.one_minus_omega, a.inv_xi, a.ref, [&](auto ic, T v) {
        st_stream(outgoing_ptr<Q, decltype(ic)::value, T, WALLS, STATE>(a.Hdst, N, nb), v);
    });
    a.Cdst[idx] = phi;
}

template <typename T, int Q, bool WALLS, int STATE>
static void launch_phase_coll(int collision, const Launch& l, const PhaseArgs<T>& a)
{
    if (collision == PHASE_SRT) phase_kernel<T, Q, WALLS, STATE, PHASE_SRT><<<l.grid, l.block, 0, l.stream>>>(a);
    else phase_kernel<T, Q, WALLS, STATE, PHASE_MRT><<<l.grid, l.block, 0, l.stream>>>(a);
}

template <typename T, int Q, bool WALLS>
static void launch_phase_state(int state, int collision, const Launch& l, const PhaseArgs<T>& a)
{
    if (a.Hpeer.lo) {      // peer mode of a slab: two-grid storage only
        if (collision == PHASE_SRT) phase_kernel<T, Q, WALLS, ST_POST, PHASE_SRT, true><<<l.grid, l.block, 0, l.stream>>>(a);
        else phase_kernel<T, Q, WALLS, ST_POST, PHASE_MRT, true><<<l.grid, l.block, 0, l.stream>>>(a);
        return;
    }
    if (state == ST_POST) launch_phase_coll<T, Q, WALLS, ST_POST>(collision, l, a);
    else if (state == ST_IN) launch_phase_coll<T, Q, WALLS, ST_IN>(collision, l, a);
    else launch_phase_coll<T, Q, WALLS, ST_SWAP>(collision, l, a);
}

template <typename T, int Q>
static void launch_phase_q(bool walls, int state, int collision, const Launch& l, const PhaseArgs<T>& a)
{
    if (walls) launch_phase_state<T, Q, true>(state, collision, l, a);
    else launch_phase_state<T, Q, false>(state, collision, l, a);
}

template <typename T>
cudaError_t launch_phase(int Q, bool walls, int state, int collision, const Launch& l, const PhaseArgs<T>& a)
{
    if (Q == 9) launch_phase_q<T, 9>(walls, state, collision, l, a);
    else if (Q == 15) launch_phase_q<T, 15>(walls, state, collision, l, a);
    else if (Q == 19) launch_phase_q<T, 19>(walls, state, collision, l, a);
    else launch_phase_q<T, 27>(walls, state, collision, l, a);
    return cudaGetLastError();
}

template cudaError_t launch_phase<ACM_T>(int, bool, int, int, const Launch&, const PhaseArgs<ACM_T>&);

}  // namespace acm
