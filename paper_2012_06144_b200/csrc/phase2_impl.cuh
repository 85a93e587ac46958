// phase2_impl.cuh -- the fused phase-field LB kernel with TWO x-adjacent cells per thread (pair.cuh, vec2.cuh) and
// its launcher, instantiated for one scalar type per translation unit (phase2_f32.cu, phase2_f64.cu).  Same
// arithmetic as phase_kernel (lb_math.cuh is shared), same storage states, walls and peer mode.
#include "kernels.h"
#include "lb_math.cuh"
#include "pair.cuh"

#ifndef ACM_PAIR_MINB
#define ACM_PAIR_MINB 1
#endif

namespace acm {

template <typename S, int Q, bool WALLS, int STATE, int COLL, bool PEER = false>
__global__ void __launch_bounds__(ACM_MAXT, ACM_PAIR_MINB) phase_kernel2(const PhaseArgs<S> a)
{
    using V = vec2<S>;
    int x0, y, z;
    if (!pair_of_thread(a.g, x0, y, z)) return;
    Nbr2 nb;
    nb.setup<WALLS>(a.g, x0, y, z);
    const unsigned idx = nb.own();
    const size_t N = a.N;      // zero-extended 32-bit value

    V h[Q];
    load_incoming2<Q, S, WALLS, STATE, PEER>(a.Hsrc, N, nb, h, a.Hpeer);
    const V ux = ldg_pair(a.U + idx), uy = ldg_pair(a.U + N + idx), uz = ldg_pair(a.U + 2 * N + idx);
    const V c0 = ldg_pair(a.Csrc + idx);
    V gx, gy, gz, lap_unused;
    fd_phi_acc<Q, V, false>(PhiGlobal2<S, PEER>{a.Csrc, &nb, a.Cpeer}, c0, gx, gy, gz, lap_unused);

    Moments<Q, V, false> m;
    m.compute(h);
    const V phi = m.m0;

    phase_collide<V, Q, COLL>(h, m, c0, gx, gy, gz, ux, uy, uz, V(a.one_minus_omega), V(a.inv_xi), V(a.ref), [&](auto ic, V v) {
        store_outgoing2<Q, decltype(ic)::value, S, WALLS, STATE>(a.Hdst, N, nb, v);
    });
    st_pair(a.Cdst + idx, phi);
}

template <typename S, int Q, bool WALLS, int STATE>
static void launch_phase2_coll(int collision, const Launch& l, const PhaseArgs<S>& a)
{
    if (collision == PHASE_SRT) phase_kernel2<S, Q, WALLS, STATE, PHASE_SRT><<<l.grid, l.block, 0, l.stream>>>(a);
    else phase_kernel2<S, Q, WALLS, STATE, PHASE_MRT><<<l.grid, l.block, 0, l.stream>>>(a);
}

template <typename S, int Q, bool WALLS>
static void launch_phase2_state(int state, int collision, const Launch& l, const PhaseArgs<S>& a)
{
    if (a.Hpeer.lo) {      // peer mode of a slab: two-grid storage only
        if (collision == PHASE_SRT) phase_kernel2<S, Q, WALLS, ST_POST, PHASE_SRT, true><<<l.grid, l.block, 0, l.stream>>>(a);
        else phase_kernel2<S, Q, WALLS, ST_POST, PHASE_MRT, true><<<l.grid, l.block, 0, l.stream>>>(a);
        return;
    }
    if (state == ST_POST) launch_phase2_coll<S, Q, WALLS, ST_POST>(collision, l, a);
    else if (state == ST_IN) launch_phase2_coll<S, Q, WALLS, ST_IN>(collision, l, a);
    else launch_phase2_coll<S, Q, WALLS, ST_SWAP>(collision, l, a);
}

template <typename S, int Q>
static void launch_phase2_q(bool walls, int state, int collision, const Launch& l, const PhaseArgs<S>& a)
{
    if (walls) launch_phase2_state<S, Q, true>(state, collision, l, a);
    else launch_phase2_state<S, Q, false>(state, collision, l, a);
}

template <typename S>
cudaError_t launch_phase2(int Q, bool walls, int state, int collision, const Launch& l, const PhaseArgs<S>& a)
{
    if (Q == 9) launch_phase2_q<S, 9>(walls, state, collision, l, a);
    else if (Q == 15) launch_phase2_q<S, 15>(walls, state, collision, l, a);
    else if (Q == 19) launch_phase2_q<S, 19>(walls, state, collision, l, a);
    else launch_phase2_q<S, 27>(walls, state, collision, l, a);
    return cudaGetLastError();
}

template cudaError_t launch_phase2<ACM_T>(int, bool, int, int, const Launch&, const PhaseArgs<ACM_T>&);

}  // namespace acm
