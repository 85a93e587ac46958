// hydro2_impl.cuh -- the fused hydrodynamic LB kernel with TWO x-adjacent cells per thread (pair.cuh, vec2.cuh) and
// its launcher, instantiated for one scalar type per translation unit (hydro2_f32.cu, hydro2_f64.cu).  Same
// arithmetic as hydro_kernel (lb_math.cuh is shared), same storage states, walls, peer mode and operator variants.
#include "kernels.h"
#include "lb_math.cuh"
#include "pair.cuh"

#ifndef ACM_PAIR_MINB
#define ACM_PAIR_MINB 1
#endif

namespace acm {

template <typename S, int Q, bool WALLS, int STATE, bool PEER = false, int HVAR = 0>
__global__ void __launch_bounds__(ACM_MAXT, ACM_PAIR_MINB) hydro_kernel2(const HydroArgs<S> a)
{
    using V = vec2<S>;
    int x0, y, z;
    if (!pair_of_thread(a.g, x0, y, z)) return;
    Nbr2 nb;
    nb.setup<WALLS>(a.g, x0, y, z);
    const unsigned idx = nb.own();
    const size_t N = a.N;      // zero-extended 32-bit value

    V g[Q];
    load_incoming2<Q, S, WALLS, STATE, PEER>(a.Gsrc, N, nb, g, a.Gpeer);
    const V uox = ld_pair(a.U + idx), uoy = ld_pair(a.U + N + idx), uoz = ld_pair(a.U + 2 * N + idx);
    const V c0 = ldg_pair(a.C + idx);
    V gpx, gpy, gpz, lap;
    fd_phi_acc<Q, V, true>(PhiGlobal2<S, PEER>{a.C, &nb, a.Cpeer}, c0, gpx, gpy, gpz, lap);

    Moments<Q, V, true> m;
    m.compute(g);
    const HydroCell<V> hc = hydro_velocity<V, Q, HVAR>(m, c0, gpx, gpy, gpz, lap, uox, uoy, uoz, a);
    st_pair(a.U + idx, hc.ux); st_pair(a.U + N + idx, hc.uy); st_pair(a.U + 2 * N + idx, hc.uz);
    hydro_collide<V, Q, HVAR>(m, hc, a, [&](auto ic, V v) {
        store_outgoing2<Q, decltype(ic)::value, S, WALLS, STATE>(a.Gdst, N, nb, v);
    });
}

template <typename S, int Q, bool WALLS>
static void launch_hydro2_state(int state, const Launch& l, const HydroArgs<S>& a)
{
    if (a.Gpeer.lo) {      // peer mode of a slab: two-grid storage only
        hydro_kernel2<S, Q, WALLS, ST_POST, true><<<l.grid, l.block, 0, l.stream>>>(a);
        return;
    }
    if (a.bulk_one || a.subiter > 1) {      // operator variants
        if (state == ST_POST) hydro_kernel2<S, Q, WALLS, ST_POST, false, 1><<<l.grid, l.block, 0, l.stream>>>(a);
        else if (state == ST_IN) hydro_kernel2<S, Q, WALLS, ST_IN, false, 1><<<l.grid, l.block, 0, l.stream>>>(a);
        else hydro_kernel2<S, Q, WALLS, ST_SWAP, false, 1><<<l.grid, l.block, 0, l.stream>>>(a);
        return;
    }
    if (state == ST_POST) hydro_kernel2<S, Q, WALLS, ST_POST><<<l.grid, l.block, 0, l.stream>>>(a);
    else if (state == ST_IN) hydro_kernel2<S, Q, WALLS, ST_IN><<<l.grid, l.block, 0, l.stream>>>(a);
    else hydro_kernel2<S, Q, WALLS, ST_SWAP><<<l.grid, l.block, 0, l.stream>>>(a);
}

template <typename S, int Q>
static void launch_hydro2_q(bool walls, int state, const Launch& l, const HydroArgs<S>& a)
{
    if (walls) launch_hydro2_state<S, Q, true>(state, l, a);
    else launch_hydro2_state<S, Q, false>(state, l, a);
}

template <typename S>
cudaError_t launch_hydro2(int Q, bool walls, int state, const Launch& l, const HydroArgs<S>& a)
{
    if (Q == 9) launch_hydro2_q<S, 9>(walls, state, l, a);
    else if (Q == 15) launch_hydro2_q<S, 15>(walls, state, l, a);
    else if (Q == 19) launch_hydro2_q<S, 19>(walls, state, l, a);
    else launch_hydro2_q<S, 27>(walls, state, l, a);
    return cudaGetLastError();
}

template cudaError_t launch_hydro2<ACM_T>(int, bool, int, const Launch&, const HydroArgs<ACM_T>&);

}  // namespace acm
