// unfused_impl.cuh -- Algorithm 1 of the paper: the "straightforward" time step made of
// six kernels -- collide h, collide g, stream h, update phi, stream g, update u -- kept as a measured
// comparison for the fusion claim of section 5 (211 -> 550 MLUPS on a P100).  Every population
// array is loaded three times and stored twice per step instead of once each.
//
// The kernels call the same per-cell device functions as the fused kernels (lb_math.cuh) and run in
// an order that is a rotation, within each population family, of the paper's listing:
//     stream h -> update phi -> collide h  |  stream g -> update u -> collide g
// With the storage convention of this library (populations kept post-collision at their own cell,
// DESIGN.md 5.2) this order reproduces the trajectory of Algorithm 2 exactly, so that both algorithms
// are checked against the same oracle.  The velocity field is double-buffered here because the
// viscous force of the collision needs u of the previous step (A10) after "update u" has run.
#include "kernels.h"
#include "lb_math.cuh"

namespace acm {

// streaming step of one population set: pull from the post-collision array `src` (periodic wrap /
// half-way bounce-back) into `dst`, which then holds the incoming populations of every cell
template <typename T, int Q, bool WALLS>
__global__ void __launch_bounds__(ACM_MAXT) stream_kernel(const T* __restrict__ src, T* __restrict__ dst, Geom g, size_t N)
{
    int x, y, z;
    if (!cell_of_thread(g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    T f[Q];
    load_incoming<Q, T, WALLS, ST_POST>(src, N, nb, f);
    static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; st_stream(dst + (size_t)i * N + idx, f[i]); });
}

// "Update phase-field": phi = sum_i h_i (eq. 7)
template <typename T, int Q>
__global__ void __launch_bounds__(ACM_MAXT) phi_kernel(const T* __restrict__ H, T* __restrict__ C, Geom g, size_t N)
{
    int x, y, z;
    if (!cell_of_thread(g, x, y, z)) return;
    const int idx = (z * g.ny + y) * g.nx + x;
    T h[Q];
    static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; h[i] = ld_stream(H + (size_t)i * N + idx); });
    Moments<Q, T, false> m;
    m.compute(h);
    C[idx] = m.m0;
}

// "Perform collision of phase-field PDFs": in place on the streamed populations; reads the new phi
// (Cdst), the stencil of the old phi (Csrc) and u
template <typename T, int Q, bool WALLS, int COLL>
__global__ void __launch_bounds__(ACM_MAXT) collide_h_kernel(const PhaseArgs<T> a)
{
    int x, y, z;
    if (!cell_of_thread(a.g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(a.g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    const size_t N = a.N;      // zero-extended 32-bit value
    T h[Q];
    static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; h[i] = ld_stream(a.Hdst + (size_t)i * N + idx); });
    const T ux = __ldg(a.U + idx), uy = __ldg(a.U + N + idx), uz = __ldg(a.U + 2 * N + idx);
    const T c0 = __ldg(a.Csrc + idx);
    T gx, gy, gz, lap_unused;
    fd_phi<Q, T, false>(a.Csrc, nb, c0, gx, gy, gz, lap_unused);
    Moments<Q, T, false> m;
    m.compute(h);
    m.m0 = a.Cdst[idx];          // the phase field written by phi_kernel
    phase_collide<T, Q, COLL>(h, m, c0, gx, gy, gz, ux, uy, uz, a.one_minus_omega, a.inv_xi, a.ref, [&](auto ic, T v) {
        st_stream(a.Hdst + (size_t) decltype(ic)::value * N + idx, v);
    });
}

// "Update the velocity" (eq. 22): u_new = sum_i g_i e_i + F/(2 rho) from the streamed g, the new phi and
// the velocity of the previous step; written to the other velocity buffer
template <typename T, int Q, bool WALLS>
__global__ void __launch_bounds__(ACM_MAXT) velocity_kernel(const HydroArgs<T> a, const T* __restrict__ Uold, T* __restrict__ Unew)
{
    int x, y, z;
    if (!cell_of_thread(a.g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(a.g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    const size_t N = a.N;      // zero-extended 32-bit value
    T g[Q];
    static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; g[i] = ld_stream(a.Gdst + (size_t)i * N + idx); });
    const T uox = Uold[idx], uoy = Uold[N + idx], uoz = Uold[2 * N + idx];
    const T c0 = __ldg(a.C + idx);
    T gpx, gpy, gpz, lap;
    fd_phi<Q, T, true>(a.C, nb, c0, gpx, gpy, gpz, lap);
    Moments<Q, T, true> m;
    m.compute(g);
    const HydroCell<T> hc = hydro_velocity<T, Q>(m, c0, gpx, gpy, gpz, lap, uox, uoy, uoz, a);
    Unew[idx] = hc.ux; Unew[N + idx] = hc.uy; Unew[2 * N + idx] = hc.uz;
}

// "Perform collision of velocity PDFs": in place on the streamed populations; evaluates the forces again
// (with u of the previous step) and takes u_new from the velocity field
template <typename T, int Q, bool WALLS>
__global__ void __launch_bounds__(ACM_MAXT) collide_g_kernel(const HydroArgs<T> a, const T* __restrict__ Uold, const T* __restrict__ Unew)
{
    int x, y, z;
    if (!cell_of_thread(a.g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(a.g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    const size_t N = a.N;      // zero-extended 32-bit value
    T g[Q];
    static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; g[i] = ld_stream(a.Gdst + (size_t)i * N + idx); });
    const T uox = Uold[idx], uoy = Uold[N + idx], uoz = Uold[2 * N + idx];
    const T c0 = __ldg(a.C + idx);
    T gpx, gpy, gpz, lap;
    fd_phi<Q, T, true>(a.C, nb, c0, gpx, gpy, gpz, lap);
    Moments<Q, T, true> m;
    m.compute(g);
    HydroCell<T> hc = hydro_velocity<T, Q>(m, c0, gpx, gpy, gpz, lap, uox, uoy, uoz, a);
    hc.ux = Unew[idx]; hc.uy = Unew[N + idx]; hc.uz = Unew[2 * N + idx];
    hydro_collide<T, Q>(m, hc, a, [&](auto ic, T v) { st_stream(a.Gdst + (size_t) decltype(ic)::value * N + idx, v); });
}

// ---- launchers ------------------------------------------------------------------------------
template <typename T, int Q, bool WALLS>
static cudaError_t unfused_phase_qw(int collision, const Launch& l, const PhaseArgs<T>& a)
{
    stream_kernel<T, Q, WALLS><<<l.grid, l.block, 0, l.stream>>>(a.Hsrc, a.Hdst, a.g, a.N);
    phi_kernel<T, Q><<<l.grid, l.block, 0, l.stream>>>(a.Hdst, a.Cdst, a.g, a.N);
    if (collision == PHASE_SRT) collide_h_kernel<T, Q, WALLS, PHASE_SRT><<<l.grid, l.block, 0, l.stream>>>(a);
    else collide_h_kernel<T, Q, WALLS, PHASE_MRT><<<l.grid, l.block, 0, l.stream>>>(a);
    return cudaGetLastError();
}

template <typename T, int Q, bool WALLS>
static cudaError_t unfused_hydro_qw(const Launch& l, const HydroArgs<T>& a, const T* Uold, T* Unew)
{
    stream_kernel<T, Q, WALLS><<<l.grid, l.block, 0, l.stream>>>(a.Gsrc, a.Gdst, a.g, a.N);
    velocity_kernel<T, Q, WALLS><<<l.grid, l.block, 0, l.stream>>>(a, Uold, Unew);
    collide_g_kernel<T, Q, WALLS><<<l.grid, l.block, 0, l.stream>>>(a, Uold, Unew);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_unfused_phase(int Q, bool walls, int collision, const Launch& l, const PhaseArgs<T>& a)
{
    if (Q == 9) return walls ? unfused_phase_qw<T, 9, true>(collision, l, a) : unfused_phase_qw<T, 9, false>(collision, l, a);
    if (Q == 15) return walls ? unfused_phase_qw<T, 15, true>(collision, l, a) : unfused_phase_qw<T, 15, false>(collision, l, a);
    if (Q == 19) return walls ? unfused_phase_qw<T, 19, true>(collision, l, a) : unfused_phase_qw<T, 19, false>(collision, l, a);
    return walls ? unfused_phase_qw<T, 27, true>(collision, l, a) : unfused_phase_qw<T, 27, false>(collision, l, a);
}

template <typename T>
cudaError_t launch_unfused_hydro(int Q, bool walls, const Launch& l, const HydroArgs<T>& a, const T* Uold, T* Unew)
{
    if (Q == 9) return walls ? unfused_hydro_qw<T, 9, true>(l, a, Uold, Unew) : unfused_hydro_qw<T, 9, false>(l, a, Uold, Unew);
    if (Q == 15) return walls ? unfused_hydro_qw<T, 15, true>(l, a, Uold, Unew) : unfused_hydro_qw<T, 15, false>(l, a, Uold, Unew);
    if (Q == 19) return walls ? unfused_hydro_qw<T, 19, true>(l, a, Uold, Unew) : unfused_hydro_qw<T, 19, false>(l, a, Uold, Unew);
    return walls ? unfused_hydro_qw<T, 27, true>(l, a, Uold, Unew) : unfused_hydro_qw<T, 27, false>(l, a, Uold, Unew);
}

template cudaError_t launch_unfused_phase<ACM_T>(int, bool, int, const Launch&, const PhaseArgs<ACM_T>&);
template cudaError_t launch_unfused_hydro<ACM_T>(int, bool, const Launch&, const HydroArgs<ACM_T>&, const ACM_T*, ACM_T*);

}  // namespace acm
