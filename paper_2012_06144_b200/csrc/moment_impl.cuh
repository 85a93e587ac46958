// moment_impl.cuh -- the two fused LB kernels in MOMENT REPRESENTATION (ACM_OPT_MOMENTS), with their initialiser and
// export kernels; instantiated for one element type per translation unit (moment_f64.cu).
//
// Both closed-form collisions produce populations of the form f*_i = w_i [A + e_i.b + e_i e_i : T] (lb_math.cuh,
// DESIGN.md 5.1): every moment of h beyond the first order and of g beyond the second order relaxes with rate 1
// (P:83), so a cell's post-collision state IS those coefficients.  This mode stores them instead of the
// populations and rebuilds, in the pull of the next step, the one population each neighbour contributes:
//   hydrodynamic step: K[10][N] = A, b (3), T (6) of g*                      (instead of Q_g populations)
//   phase-field step:  M[4][N]  = A, b (3) of h*; its T = 4.5 phi u u^T is rebuilt from phi and the velocity the
//                      collision used, which is still there because u is double-buffered in this mode
// The trajectory is the one of the population kernels up to rounding (same oracle, same bars); what changes is the
// traffic: 8 (11 + 5) = 128 B (phase) + 8 (14 + 13) = 216 B (hydro) per cell and step for every lattice, instead of
// 280 + 360 B (D3Q15 + D3Q19) or 472 + 488 B (D3Q27 + D3Q27).  The price is the gather: a pulled population needs up
// to 6 (g) / 8 (h) values of the neighbour instead of one, served by L1/L2.
#include "kernels.h"
#include "lb_math.cuh"

namespace acm {

// index of the cell that delivers population I to the calling cell, and whether the delivery is a bounce-back
// (then the cell itself delivers its own opposite population: same even part, odd part with the other sign)
template <int Q, int I, bool WALLS, bool LOCAL>
__device__ __forceinline__ unsigned mom_source(const Nbr& nb, bool& flip)
{
    using L = Lat<Q>;
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I);
    flip = false;
    if constexpr (LOCAL || I == 0) return nb.at<0, 0, 0>();
    else {
        if constexpr (WALLS) {
            if (nb.template beyond<-ex, -ey, -ez, WALLS>()) { flip = true; return nb.at<0, 0, 0>(); }
        }
        return nb.template at<-ex, -ey, -ez>();
    }
}

// s * v with s in {-1, 0, 1} known at compile time, accumulated into acc (first = nothing accumulated yet)
template <int S, typename T>
__device__ __forceinline__ void odd_term(T& acc, bool& first, T v)
{
    if constexpr (S != 0) {
        if (first) { acc = S > 0 ? v : -v; first = false; }
        else addsgn<S>(acc, v);
    }
}

// incoming hydrodynamic population g_I(x) / w_I rebuilt from the coefficient array K[10][N].
// LOCAL: K holds the coefficients of the cell's own INCOMING populations (state right after acm_init, whose g is
// defined pre-collision at its cell, A13/A14): no streaming.
template <int Q, int I, typename T, bool WALLS, bool LOCAL>
__device__ __forceinline__ T mom_pull_g(const T* __restrict__ K, size_t N, const Nbr& nb)
{
    using L = Lat<Q>;
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I);
    bool flip;
    const unsigned j = mom_source<Q, I, WALLS, LOCAL>(nb, flip);
    const T* k = K + j;
    T E = __ldg(k);                                              // A
    if constexpr (ex != 0) E += __ldg(k + 4 * N);                // e e : T, diagonal part
    if constexpr (ey != 0) E += __ldg(k + 5 * N);
    if constexpr (ez != 0) E += __ldg(k + 6 * N);
    if constexpr (ex * ey != 0) E += T(2 * ex * ey) * __ldg(k + 7 * N);
    if constexpr (ex * ez != 0) E += T(2 * ex * ez) * __ldg(k + 8 * N);
    if constexpr (ey * ez != 0) E += T(2 * ey * ez) * __ldg(k + 9 * N);
    if constexpr (I == 0) return E;
    else {
        T O = T(0);
        bool first = true;
        if constexpr (ex != 0) odd_term<ex>(O, first, __ldg(k + 1 * N));
        if constexpr (ey != 0) odd_term<ey>(O, first, __ldg(k + 2 * N));
        if constexpr (ez != 0) odd_term<ez>(O, first, __ldg(k + 3 * N));
        if constexpr (WALLS) return flip ? E - O : E + O;
        else return E + O;
    }
}

// incoming phase-field population h_I(x) / w_I rebuilt from M[4][N] (A, b), phi and the velocity Uo the collision
// that wrote M used:  h*_i = w_i [A + e_i.b + 4.5 phi (e_i.u)^2],  A = phi (1 - 1.5 u^2),  b = 3 phi u + F-part + relaxed part
template <int Q, int I, typename T, bool WALLS, bool LOCAL = false>
__device__ __forceinline__ T mom_pull_h(const T* __restrict__ M, const T* __restrict__ C, const T* __restrict__ Uo, size_t N,
                                        const Nbr& nb)
{
    using L = Lat<Q>;
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I);
    bool flip;
    const unsigned j = mom_source<Q, I, WALLS, LOCAL>(nb, flip);
    const T* m = M + j;
    const T A = __ldg(m);
    if constexpr (I == 0) return A;
    else {
        T O = T(0), eu = T(0);
        bool fo = true, fu = true;
        if constexpr (ex != 0) { odd_term<ex>(O, fo, __ldg(m + 1 * N)); odd_term<ex>(eu, fu, __ldg(Uo + j)); }
        if constexpr (ey != 0) { odd_term<ey>(O, fo, __ldg(m + 2 * N)); odd_term<ey>(eu, fu, __ldg(Uo + N + j)); }
        if constexpr (ez != 0) { odd_term<ez>(O, fo, __ldg(m + 3 * N)); odd_term<ez>(eu, fu, __ldg(Uo + 2 * N + j)); }
        const T E = A + T(4.5) * __ldg(C + j) * (eu * eu);
        if constexpr (WALLS) return flip ? E - O : E + O;
        else return E + O;
    }
}

// ------------------------------------------------------------------------------------------
// Kernel 1 in moment representation (Alg. 2; eqs. 4-7, 23)
// ------------------------------------------------------------------------------------------
template <typename T, int Q, bool WALLS>
__global__ void __launch_bounds__(ACM_MAXT) phase_mom_kernel(const MomPhaseArgs<T> a)
{
    int x, y, z;
    if (!cell_of_thread(a.g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(a.g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    const size_t N = a.N;

    T h[Q];
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        h[i] = T(Lat<Q>::w(i)) * mom_pull_h<Q, i, T, WALLS>(a.Msrc, a.Csrc, a.Uold, N, nb);
    });
    const T ux = __ldg(a.U + idx), uy = __ldg(a.U + N + idx), uz = __ldg(a.U + 2 * N + idx);
    const T c0 = __ldg(a.Csrc + idx);
    T gx, gy, gz, lap_unused;
    fd_phi<Q, T, false>(a.Csrc, nb, c0, gx, gy, gz, lap_unused);

    Moments<Q, T, false> m;
    m.compute(h);
    const T phi = m.m0;
    // the MRT branch of phase_collide (lb_math.cuh) up to the coefficients
    const T g2 = gx * gx + gy * gy + gz * gz;
    const T inv = inv_norm_or_zero(g2);
    const T dc = c0 - T(0.5);
    const T theta = (T(1) - T(4) * dc * dc) * a.inv_xi;
    const T tnx = theta * inv * gx, tny = theta * inv * gy, tnz = theta * inv * gz;
    const T k = T(3) * a.one_minus_omega;
    const T sixth = T(1.0 / 6.0);
    const T dxm = m.jx - phi * ux + sixth * tnx;
    const T dym = m.jy - phi * uy + sixth * tny;
    const T dzm = m.jz - phi * uz + sixth * tnz;
    const T p3 = T(3) * phi;
    const T usq = T(1.5) * (ux * ux + uy * uy + uz * uz);
    a.Mdst[idx] = phi * (T(1) - usq);
    a.Mdst[N + idx] = p3 * ux + T(0.5) * tnx + k * dxm;
    a.Mdst[2 * N + idx] = p3 * uy + T(0.5) * tny + k * dym;
    a.Mdst[3 * N + idx] = p3 * uz + T(0.5) * tnz + k * dzm;
    a.Cdst[idx] = phi;
}

// ------------------------------------------------------------------------------------------
// Kernel 2 in moment representation (Alg. 2; eqs. 8, 10-22, 24, 25, 30)
// ------------------------------------------------------------------------------------------
template <typename T, int Q, bool WALLS, bool LOCAL, int HVAR>
__global__ void __launch_bounds__(ACM_MAXT) hydro_mom_kernel(const MomHydroArgs<T> a)
{
    int x, y, z;
    if (!cell_of_thread(a.h.g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(a.h.g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    const size_t N = a.h.N;

    T g[Q];
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        g[i] = T(Lat<Q>::w(i)) * mom_pull_g<Q, i, T, WALLS, LOCAL>(a.Ksrc, N, nb);
    });
    const T uox = __ldg(a.Uin + idx), uoy = __ldg(a.Uin + N + idx), uoz = __ldg(a.Uin + 2 * N + idx);
    const T c0 = __ldg(a.h.C + idx);
    T gpx, gpy, gpz, lap;
    fd_phi<Q, T, true>(a.h.C, nb, c0, gpx, gpy, gpz, lap);

    Moments<Q, T, true> m;
    m.compute(g);
    const HydroCell<T> hc = hydro_velocity<T, Q, HVAR>(m, c0, gpx, gpy, gpz, lap, uox, uoy, uoz, a.h);
    a.Uout[idx] = hc.ux; a.Uout[N + idx] = hc.uy; a.Uout[2 * N + idx] = hc.uz;
    const Coeffs<T> k = hydro_coeffs<T, Q, HVAR>(m, hc, a.h);
    T* o = a.Kdst + idx;
    o[0] = k.A; o[N] = k.bx; o[2 * N] = k.by; o[3 * N] = k.bz;
    o[4 * N] = k.Txx; o[5 * N] = k.Tyy; o[6 * N] = k.Tzz; o[7 * N] = k.Txy; o[8 * N] = k.Txz; o[9 * N] = k.Tyz;
}

// ------------------------------------------------------------------------------------------
// Equilibrium initialiser (Alg. 2 line 1): phi, u (both velocity buffers), the coefficients of h* = phi Gamma(u)
// (post-collision convention: the first phase-field step streams it) and of the INCOMING g = Gamma(u) - w (the first
// hydrodynamic step collides it where it is: hydro_mom_kernel<LOCAL>).
// ------------------------------------------------------------------------------------------
template <typename T>
__global__ void init_mom_kernel(const T* __restrict__ phi, const T* __restrict__ u, T* M, T* K, T* C, T* U0, T* U1, Geom g, size_t N)
{
    int x, y, z;
    if (!cell_of_thread(g, x, y, z)) return;
    const size_t idx = ((size_t)z * g.ny + y) * g.nx + x;
    const T ph = phi[idx];
    const T ux = u[idx], uy = u[N + idx], uz = u[2 * N + idx];
    C[idx] = ph;
    U0[idx] = ux; U0[N + idx] = uy; U0[2 * N + idx] = uz;
    U1[idx] = ux; U1[N + idx] = uy; U1[2 * N + idx] = uz;
    const T usq = T(1.5) * (ux * ux + uy * uy + uz * uz);
    M[idx] = ph * (T(1) - usq);
    M[N + idx] = T(3) * ph * ux; M[2 * N + idx] = T(3) * ph * uy; M[3 * N + idx] = T(3) * ph * uz;
    T* k = K + idx;
    k[0] = -usq;
    k[N] = T(3) * ux; k[2 * N] = T(3) * uy; k[3 * N] = T(3) * uz;
    k[4 * N] = T(4.5) * ux * ux; k[5 * N] = T(4.5) * uy * uy; k[6 * N] = T(4.5) * uz * uz;
    k[7 * N] = T(4.5) * ux * uy; k[8 * N] = T(4.5) * ux * uz; k[9 * N] = T(4.5) * uy * uz;
}

// Export in the ABI's conventions: h post-collision at its own cell (rebuilt locally), g incoming (the pending pull
// applied); optionally p = c_s^2 rho(phi) sum_i g_i.
template <typename T, int Q>
__global__ void export_h_mom_kernel(const T* __restrict__ M, const T* __restrict__ C, const T* __restrict__ Uo, T* out, Geom g, size_t N)
{
    int x, y, z;
    if (!cell_of_thread(g, x, y, z)) return;
    Nbr nb;
    nb.setup<true>(g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        out[(size_t)i * N + idx] = T(Lat<Q>::w(i)) * mom_pull_h<Q, i, T, false, true>(M, C, Uo, N, nb);
    });
}

template <typename T, int Q, bool LOCAL>
__global__ void export_g_mom_kernel(const T* __restrict__ K, const T* __restrict__ C, T* out, T* p, Geom g, size_t N, T rho_L, T drho)
{
    int x, y, z;
    if (!cell_of_thread(g, x, y, z)) return;
    Nbr nb;
    nb.setup<true>(g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    T f[Q];
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        f[i] = T(Lat<Q>::w(i)) * mom_pull_g<Q, i, T, true, LOCAL>(K, N, nb);
    });
    if (out) static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; out[(size_t)i * N + idx] = f[i]; });
    if (p) {
        Moments<Q, T, false> m;
        m.compute(f);
        p[idx] = m.m0 * (rho_L + C[idx] * drho) * T(1.0 / 3.0);
    }
}

// ------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------
#define ACM_MOM_DISPATCH_Q(q, QQ, ...)                              \
    switch (q) {                                                    \
        case 9: { constexpr int QQ = 9; __VA_ARGS__; } break;       \
        case 15: { constexpr int QQ = 15; __VA_ARGS__; } break;     \
        case 19: { constexpr int QQ = 19; __VA_ARGS__; } break;     \
        default: { constexpr int QQ = 27; __VA_ARGS__; } break;     \
    }

template <typename T>
cudaError_t launch_phase_mom(int Q, bool walls, const Launch& l, const MomPhaseArgs<T>& a)
{
    ACM_MOM_DISPATCH_Q(Q, QQ, {
        if (walls) phase_mom_kernel<T, QQ, true><<<l.grid, l.block, 0, l.stream>>>(a);
        else phase_mom_kernel<T, QQ, false><<<l.grid, l.block, 0, l.stream>>>(a);
    });
    return cudaGetLastError();
}

template <typename T, int Q, bool WALLS>
static void launch_hydro_mom_q(bool local, const Launch& l, const MomHydroArgs<T>& a)
{
    const bool var = a.h.bulk_one || a.h.subiter > 1;
    if (local) {
        if (var) hydro_mom_kernel<T, Q, WALLS, true, 1><<<l.grid, l.block, 0, l.stream>>>(a);
        else hydro_mom_kernel<T, Q, WALLS, true, 0><<<l.grid, l.block, 0, l.stream>>>(a);
    } else {
        if (var) hydro_mom_kernel<T, Q, WALLS, false, 1><<<l.grid, l.block, 0, l.stream>>>(a);
        else hydro_mom_kernel<T, Q, WALLS, false, 0><<<l.grid, l.block, 0, l.stream>>>(a);
    }
}

template <typename T>
cudaError_t launch_hydro_mom(int Q, bool walls, bool local, const Launch& l, const MomHydroArgs<T>& a)
{
    ACM_MOM_DISPATCH_Q(Q, QQ, {
        if (walls) launch_hydro_mom_q<T, QQ, true>(local, l, a);
        else launch_hydro_mom_q<T, QQ, false>(local, l, a);
    });
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_init_mom(const Launch& l, const T* phi, const T* u, T* M, T* K, T* C, T* U0, T* U1, Geom g, size_t N)
{
    init_mom_kernel<T><<<l.grid, l.block, 0, l.stream>>>(phi, u, M, K, C, U0, U1, g, N);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_export_h_mom(int Q, const Launch& l, const T* M, const T* C, const T* Uo, T* out, Geom g, size_t N)
{
    ACM_MOM_DISPATCH_Q(Q, QQ, { export_h_mom_kernel<T, QQ><<<l.grid, l.block, 0, l.stream>>>(M, C, Uo, out, g, N); });
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_export_g_mom(int Q, bool local, const Launch& l, const T* K, const T* C, T* out, T* p, Geom g, size_t N, T rho_L, T drho)
{
    ACM_MOM_DISPATCH_Q(Q, QQ, {
        if (local) export_g_mom_kernel<T, QQ, true><<<l.grid, l.block, 0, l.stream>>>(K, C, out, p, g, N, rho_L, drho);
        else export_g_mom_kernel<T, QQ, false><<<l.grid, l.block, 0, l.stream>>>(K, C, out, p, g, N, rho_L, drho);
    });
    return cudaGetLastError();
}

template cudaError_t launch_phase_mom<ACM_T>(int, bool, const Launch&, const MomPhaseArgs<ACM_T>&);
template cudaError_t launch_hydro_mom<ACM_T>(int, bool, bool, const Launch&, const MomHydroArgs<ACM_T>&);
template cudaError_t launch_init_mom<ACM_T>(const Launch&, const ACM_T*, const ACM_T*, ACM_T*, ACM_T*, ACM_T*, ACM_T*, ACM_T*, Geom, size_t);
template cudaError_t launch_export_h_mom<ACM_T>(int, const Launch&, const ACM_T*, const ACM_T*, const ACM_T*, ACM_T*, Geom, size_t);
template cudaError_t launch_export_g_mom<ACM_T>(int, bool, const Launch&, const ACM_T*, const ACM_T*, ACM_T*, ACM_T*, Geom, size_t, ACM_T, ACM_T);

}  // namespace acm
