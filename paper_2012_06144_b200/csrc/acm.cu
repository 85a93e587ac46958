// acm.cu -- libacm: hand-written sm_100a CUDA kernels for the coupled ACM lattice-Boltzmann step
// of arXiv 2012.06144 and the C ABI of include/acm.h.  See DESIGN.md for the data layout, the
// closed-form collisions and the byte accounting.  Shares no code with oracle/.
//
// Storage on the device (all SoA, x fastest, 64-bit offsets for the q planes):
//   H[2][Qh][N]  phase populations, post-collision value at their own cell (pulled by the next step)
//   G[2][Qg][N]  hydrodynamic populations, ALSO stored post-collision at their own cell: the paper's
//                "collide-stream-push" is realised as a pull at the start of the next
//                hydrodynamic step ("lazy pull"); acm_get_pdfs / acm_fields apply the pending
//                streaming, the initialiser pre-shifts g.  Aligned, fully coalesced stores.
//   C[2][N]      phi (double-buffered: the phase kernel reads a stencil of the old phi and writes new)
//   U[3][N]      velocity, in place
#include <cuda_runtime.h>
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/acm.h"
#include "lattice.cuh"

namespace acm {

// ------------------------------------------------------------------------------------------
// geometry: neighbour indexing with periodic wrap, wall flags for half-way bounce-back
// ------------------------------------------------------------------------------------------
struct Geom {
    int nx, ny, nz;
    unsigned walls;
};

// Per-cell neighbourhood: coordinates of x-1, x, x+1 (periodic wrap; clamped at a wall, which is
// the mirror ghost phi(x,-1,z) = phi(x,0,z) of the FD stencils) and "beyond a wall" flags.
struct Nbr {
    int xs[3];        // x-1, x, x+1
    int row[3][3];    // [dz+1][dy+1] -> (z'*ny + y')*nx
    bool wxm, wxp, wym, wyp, wzm, wzp;   // the cell at x-1 / x+1 / ... lies beyond a wall

    template <bool WALLS>
    __device__ __forceinline__ void setup(const Geom& g, int x, int y, int z)
    {
        wxm = wxp = wym = wyp = wzm = wzp = false;
        int xm = x - 1, xp = x + 1, ym = y - 1, yp = y + 1, zm = z - 1, zp = z + 1;
        if (xm < 0) { if (WALLS && (g.walls & ACM_WALL_X)) { wxm = true; xm = 0; } else xm = g.nx - 1; }
        if (xp >= g.nx) { if (WALLS && (g.walls & ACM_WALL_X)) { wxp = true; xp = g.nx - 1; } else xp = 0; }
        if (ym < 0) { if (WALLS && (g.walls & ACM_WALL_Y)) { wym = true; ym = 0; } else ym = g.ny - 1; }
        if (yp >= g.ny) { if (WALLS && (g.walls & ACM_WALL_Y)) { wyp = true; yp = g.ny - 1; } else yp = 0; }
        if (zm < 0) { if (WALLS && (g.walls & ACM_WALL_Z)) { wzm = true; zm = 0; } else zm = g.nz - 1; }
        if (zp >= g.nz) { if (WALLS && (g.walls & ACM_WALL_Z)) { wzp = true; zp = g.nz - 1; } else zp = 0; }
        xs[0] = xm; xs[1] = x; xs[2] = xp;
        const int ys[3] = {ym, y, yp}, zs[3] = {zm, z, zp};
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) row[a][b] = (zs[a] * g.ny + ys[b]) * g.nx;
    }
    // index of the cell at offset (dx,dy,dz), each in {-1,0,1}
    template <int DX, int DY, int DZ>
    __device__ __forceinline__ int at() const { return row[DZ + 1][DY + 1] + xs[DX + 1]; }
    // is the cell at offset (dx,dy,dz) beyond a wall?
    template <int DX, int DY, int DZ, bool WALLS>
    __device__ __forceinline__ bool beyond() const
    {
        if constexpr (!WALLS) return false;
        bool b = false;
        if constexpr (DX < 0) b |= wxm;
        if constexpr (DX > 0) b |= wxp;
        if constexpr (DY < 0) b |= wym;
        if constexpr (DY > 0) b |= wyp;
        if constexpr (DZ < 0) b |= wzm;
        if constexpr (DZ > 0) b |= wzp;
        return b;
    }
};

// tuning knobs (defaults = the measured best on B200)
#ifndef ACM_LD
#define ACM_LD 2
#endif
#ifndef ACM_ST
#define ACM_ST 2
#endif
#ifndef ACM_PHASE_MINB
#define ACM_PHASE_MINB 1
#endif
#ifndef ACM_HYDRO_MINB
#define ACM_HYDRO_MINB 1
#endif
#ifndef ACM_MAXT
#define ACM_MAXT 256
#endif

// population loads/stores.  Measured on B200 (profiles/r1_variants.md): plain ld/st beat the
// streaming hints (__ldcs/__stcs) by 5 % on the whole step, so plain is the default.
template <typename T> __device__ __forceinline__ T ld_stream(const T* p)
{
#if ACM_LD == 0
    return __ldcs(p);
#elif ACM_LD == 1
    return __ldg(p);
#else
    return *p;
#endif
}
template <typename T> __device__ __forceinline__ void st_stream(T* p, T v)
{
#if ACM_ST == 0
    __stcs(p, v);
#elif ACM_ST == 1
    __stcg(p, v);
#else
    *p = v;
#endif
}

// ------------------------------------------------------------------------------------------
// Storage states of a population array and the streaming they imply.
//   ST_POST  (two-grid): slot i at x holds the post-collision f*_i(x); the next step pulls.
//   ST_IN    (in place): slot i at x holds the incoming (streamed, pre-collision) f_i(x).
//   ST_SWAP  (in place): slot ibar at x holds the post-collision f*_i(x) (directions swapped).
// Two-grid update: ST_POST(src) -> ST_POST(dst).  In-place AA pattern (Bailey et al. 2009; the paper
// names it P:52): even step ST_IN -> ST_SWAP touches only the own cell, odd step ST_SWAP -> ST_IN
// reads slot ibar at x-e_i and writes slot i at x+e_i -- exactly the locations it read, so one array
// suffices.  Half-way bounce-back: a population that would come from / go to a cell beyond a wall is
// taken from / put into the opposite slot of the own cell.
// ------------------------------------------------------------------------------------------
enum { ST_POST = 0, ST_IN = 1, ST_SWAP = 2 };

// incoming populations f_i(x) from an array in state STATE
template <int Q, typename T, bool WALLS, int STATE>
__device__ __forceinline__ void load_incoming(const T* F, size_t N, const Nbr& nb, T (&f)[Q])
{
    using L = Lat<Q>;
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int ex = L::ex(i), ey = L::ey(i), ez = L::ez(i), o = L::opp(i);
        const T* src;
        if constexpr (STATE == ST_IN) {
            src = F + (size_t)i * N + nb.template at<0, 0, 0>();
        } else {
            constexpr int far = (STATE == ST_POST) ? i : o;      // slot at x - e_i
            constexpr int own = (STATE == ST_POST) ? o : i;      // slot at x when x - e_i is beyond a wall
            src = F + (size_t)far * N + nb.template at<-ex, -ey, -ez>();
            if constexpr (WALLS && i > 0) {
                if (nb.template beyond<-ex, -ey, -ez, WALLS>()) src = F + (size_t)own * N + nb.template at<0, 0, 0>();
            }
        }
        f[i] = ld_stream(src);
    });
}

// address of the post-collision population f*_i(x) in the array the step writes.
// FROM is the state the step read: ST_POST -> two-grid dst (ST_POST), ST_IN -> ST_SWAP, ST_SWAP -> ST_IN.
template <int Q, int I, typename T, bool WALLS, int FROM>
__device__ __forceinline__ T* outgoing_ptr(T* F, size_t N, const Nbr& nb)
{
    using L = Lat<Q>;
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I), o = L::opp(I);
    if constexpr (FROM == ST_POST) {
        return F + (size_t)I * N + nb.template at<0, 0, 0>();
    } else if constexpr (FROM == ST_IN) {
        return F + (size_t)o * N + nb.template at<0, 0, 0>();
    } else {
        T* dst = F + (size_t)I * N + nb.template at<ex, ey, ez>();
        if constexpr (WALLS && I > 0) {
            if (nb.template beyond<ex, ey, ez, WALLS>()) dst = F + (size_t)o * N + nb.template at<0, 0, 0>();
        }
        return dst;
    }
}

// post-collision population f*_i(x) read back from an array in state STATE (export only)
template <int Q, int I, typename T, int STATE>
__device__ __forceinline__ T load_post(const T* F, size_t N, const Nbr& nb)
{
    using L = Lat<Q>;
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I), o = L::opp(I);
    if constexpr (STATE == ST_POST) return F[(size_t)I * N + nb.template at<0, 0, 0>()];
    else if constexpr (STATE == ST_SWAP) return F[(size_t)o * N + nb.template at<0, 0, 0>()];
    else {
        if (nb.template beyond<ex, ey, ez, true>()) return F[(size_t)o * N + nb.template at<0, 0, 0>()];
        return F[(size_t)I * N + nb.template at<ex, ey, ez>()];
    }
}

// Isotropic finite differences of phi on lattice Q (eqs. 23, 24 with c = dx = 1, c_s^2 = 1/3):
//   grad phi = 3 sum_i w_i e_i phi(x+e_i)      (summed as opposite-pair differences)
//   lap  phi = 6 sum_i w_i [phi(x+e_i) - phi(x)]
template <int Q, typename T, bool LAPLACE>
__device__ __forceinline__ void fd_phi(const T* __restrict__ C, const Nbr& nb, T c0, T& gx, T& gy, T& gz, T& lap)
{
    using L = Lat<Q>;
    T dx[4] = {0, 0, 0, 0}, dy[4] = {0, 0, 0, 0}, dz[4] = {0, 0, 0, 0}, ss[4] = {0, 0, 0, 0};   // per class
    static_for<1, Q, 2>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int ex = L::ex(i), ey = L::ey(i), ez = L::ez(i), c = L::cls(i);
        const T p = __ldg(C + nb.template at<ex, ey, ez>());
        const T m = __ldg(C + nb.template at<-ex, -ey, -ez>());
        const T d = p - m;
        addsgn<ex>(dx[c], d); addsgn<ey>(dy[c], d); addsgn<ez>(dz[c], d);
        if constexpr (LAPLACE) ss[c] += p + m;
    });
    gx = gy = gz = T(0);
    T l = T(0), wsum = T(0);
    static_for<1, 4>([&](auto cc) {
        constexpr int c = decltype(cc)::value;
        if constexpr (L::has_cls(c)) {
            constexpr T w3 = T(3.0 * L::wc(c));
            gx += w3 * dx[c]; gy += w3 * dy[c]; gz += w3 * dz[c];
            if constexpr (LAPLACE) l += T(6.0 * L::wc(c)) * ss[c];
        }
    });
    (void)wsum;
    if constexpr (LAPLACE) lap = l - T(6.0 * (1.0 - L::wc(0))) * c0;   // sum_{i>=1} w_i = 1 - w_0
}

// ------------------------------------------------------------------------------------------
// Kernel 1: fused phase-field LB step (Alg. 2; eqs. 4-7, 23)
//   pull h -> phi_new = sum h -> grad/normal/theta from the OLD phi -> closed-form MRT collision
//   (first-order moments relaxed with omega_phi, all others with 1) -> store h, phi_new.
// With d = j - phi_new u + (theta/6) n:   h*_i = h^eq_i + F_i/2 + (1-omega_phi) 3 w_i e_i.d
// ------------------------------------------------------------------------------------------
template <typename T>
struct PhaseArgs {
    const T* Hsrc; T* Hdst;
    const T* Csrc; T* Cdst;
    const T* U;
    Geom g;
    size_t N;
    T one_minus_omega, inv_xi;
};

template <typename T, int Q, bool WALLS, int STATE>
__global__ void __launch_bounds__(ACM_MAXT, ACM_PHASE_MINB) phase_kernel(const PhaseArgs<T> a)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z * blockDim.z + threadIdx.z;
    if (x >= a.g.nx || y >= a.g.ny || z >= a.g.nz) return;
    Nbr nb;
    nb.setup<WALLS>(a.g, x, y, z);
    const int idx = nb.at<0, 0, 0>();
    const size_t N = a.N;

    T h[Q];
    load_incoming<Q, T, WALLS, STATE>(a.Hsrc, N, nb, h);
    const T ux = __ldg(a.U + idx), uy = __ldg(a.U + N + idx), uz = __ldg(a.U + 2 * N + idx);
    const T c0 = __ldg(a.Csrc + idx);
    T gx, gy, gz, lap_unused;
    fd_phi<Q, T, false>(a.Csrc, nb, c0, gx, gy, gz, lap_unused);

    Moments<Q, T, false> m;
    m.compute(h);
    const T phi = m.m0;

    // interface normal (n = 0 where grad phi vanishes exactly) and theta = (1 - 4 (phi-1/2)^2)/xi
    const T g2 = gx * gx + gy * gy + gz * gz;
    const T inv = (g2 > T(0)) ? T(1) / sqrt(g2) : T(0);
    const T dc = c0 - T(0.5);
    const T theta = (T(1) - T(4) * dc * dc) * a.inv_xi;
    const T tnx = theta * inv * gx, tny = theta * inv * gy, tnz = theta * inv * gz;   // theta * n

    const T k = T(3) * a.one_minus_omega;
    const T sixth = T(1.0 / 6.0);
    const T dxm = m.jx - phi * ux + sixth * tnx;
    const T dym = m.jy - phi * uy + sixth * tny;
    const T dzm = m.jz - phi * uz + sixth * tnz;
    const T A = phi * (T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz));
    const T p3 = T(3) * phi;
    const T bx = p3 * ux + T(0.5) * tnx + k * dxm;
    const T by = p3 * uy + T(0.5) * tny + k * dym;
    const T bz = p3 * uz + T(0.5) * tnz + k * dzm;
    const T p45 = T(4.5) * phi;
    if constexpr (sizeof(T) == 8) {
        emit_populations<Q, T>(A, bx, by, bz, p45 * ux * ux, p45 * uy * uy, p45 * uz * uz, p45 * ux * uy, p45 * ux * uz,
                               p45 * uy * uz, [&](auto ic, T v) {
                                   st_stream(outgoing_ptr<Q, decltype(ic)::value, T, WALLS, STATE>(a.Hdst, N, nb), v);
                               });
    } else {
        // fp32 instance (reading A22): the rest population is set by subtraction,
        // h*_0 = phi_new - sum_{i>=1} h*_i, so that the collision conserves phi exactly in fp32.
        T rest = phi;
        emit_populations<Q, T>(A, bx, by, bz, p45 * ux * ux, p45 * uy * uy, p45 * uz * uz, p45 * ux * uy, p45 * ux * uz,
                               p45 * uy * uz, [&](auto ic, T v) {
                                   constexpr int i = decltype(ic)::value;
                                   if constexpr (i > 0) { rest -= v; st_stream(outgoing_ptr<Q, i, T, WALLS, STATE>(a.Hdst, N, nb), v); }
                               });
        st_stream(outgoing_ptr<Q, 0, T, WALLS, STATE>(a.Hdst, N, nb), rest);
    }
    a.Cdst[idx] = phi;
}

// ------------------------------------------------------------------------------------------
// Kernel 2: fused hydrodynamic LB step (Alg. 2; eqs. 8, 10-22, 24, 25, 30)
//   pull g -> p*, j, P -> rho, tau, s_nu, grad/lap of the NEW phi, mu_phi -> F_s+F_p+F_mu+F_b ->
//   u_new = j + F/(2 rho) -> closed-form MRT collision (second-order moments relaxed with s_nu,
//   all others with 1) -> store g (own cell, see header), u_new.
//   g*_i = g^eq_i(u_new) + F_i/2 + (1 - s_nu) 4.5 w_i (e_ia e_ib - d_ab/3) Pi_ab,
//   Pi = P - p*/3 I - u_new u_new^T;  F_mu = -tau s_nu (P - p*/3 I - u_old u_old^T) grad rho
// ------------------------------------------------------------------------------------------
template <typename T>
struct HydroArgs {
    const T* Gsrc; T* Gdst;
    const T* C;      // new phi
    T* U;
    Geom g;
    size_t N;
    T rho_L, drho, tau_L, dtau, beta4, kappa, gx, gy, gz;
};

template <typename T, int Q, bool WALLS, int STATE>
__global__ void __launch_bounds__(ACM_MAXT, ACM_HYDRO_MINB) hydro_kernel(const HydroArgs<T> a)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z * blockDim.z + threadIdx.z;
    if (x >= a.g.nx || y >= a.g.ny || z >= a.g.nz) return;
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

// ------------------------------------------------------------------------------------------
// Equilibrium initialiser (Alg. 2 line 1): C <- phi, U <- u, h*_i <- phi Gamma_i(u) (post-collision
// convention: the first phase step streams it), g_i <- Gamma_i(u) - w_i (incoming convention: the
// first hydrodynamic step collides it).  Storage: two-grid keeps both sets in ST_POST, so g is
// pre-shifted (Gs_i(y) = g_i(y+e_i), or g_ibar(y) if y+e_i lies beyond a wall); in place h starts
// in ST_SWAP and g in ST_IN.
// ------------------------------------------------------------------------------------------
template <int Q, typename T>
__device__ __forceinline__ T gamma_i(int ex, int ey, int ez, T w, T ux, T uy, T uz)
{
    const T eu = T(ex) * ux + T(ey) * uy + T(ez) * uz;
    return w * (T(1) + T(3) * eu + T(4.5) * eu * eu - T(1.5) * (ux * ux + uy * uy + uz * uz));
}

template <typename T, int QH, int QG, bool INPLACE>
__global__ void init_kernel(const T* __restrict__ phi, const T* __restrict__ u, T* H, T* G, T* C, T* U, Geom g, size_t N)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z * blockDim.z + threadIdx.z;
    if (x >= g.nx || y >= g.ny || z >= g.nz) return;
    Nbr nb;
    nb.setup<true>(g, x, y, z);
    const int idx = nb.at<0, 0, 0>();
    const T ph = phi[idx];
    const T ux = u[idx], uy = u[N + idx], uz = u[2 * N + idx];
    C[idx] = ph;
    U[idx] = ux; U[N + idx] = uy; U[2 * N + idx] = uz;
    static_for<0, QH>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        using L = Lat<QH>;
        constexpr int slot = INPLACE ? L::opp(i) : i;
        H[(size_t)slot * N + idx] = ph * gamma_i<QH, T>(L::ex(i), L::ey(i), L::ez(i), T(L::w(i)), ux, uy, uz);
    });
    static_for<0, QG>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        using L = Lat<QG>;
        constexpr int ex = L::ex(i), ey = L::ey(i), ez = L::ez(i);
        T v;
        if constexpr (INPLACE) {
            v = gamma_i<QG, T>(ex, ey, ez, T(L::w(i)), ux, uy, uz) - T(L::w(i));
        } else if (nb.template beyond<ex, ey, ez, true>()) {
            constexpr int o = L::opp(i);
            v = gamma_i<QG, T>(L::ex(o), L::ey(o), L::ez(o), T(L::w(o)), ux, uy, uz) - T(L::w(o));
        } else {
            const int j = nb.template at<ex, ey, ez>();
            v = gamma_i<QG, T>(ex, ey, ez, T(L::w(i)), u[j], u[N + j], u[2 * N + j]) - T(L::w(i));
        }
        G[(size_t)i * N + idx] = v;
    });
}

// ------------------------------------------------------------------------------------------
// Diagnostics and debug export / import
// ------------------------------------------------------------------------------------------
// Export of a population array stored in state STATE, in the convention POST (post-collision value at
// its own cell) or incoming (streamed value); optionally p = c_s^2 rho(phi) sum_i f_i.
template <typename T, int Q, int STATE, bool POST>
__global__ void export_kernel(const T* F, const T* __restrict__ C, T* out, T* p, Geom g, size_t N, T rho_L, T drho)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z * blockDim.z + threadIdx.z;
    if (x >= g.nx || y >= g.ny || z >= g.nz) return;
    Nbr nb;
    nb.setup<true>(g, x, y, z);
    const int idx = nb.at<0, 0, 0>();
    T f[Q];
    if constexpr (POST) static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; f[i] = load_post<Q, i, T, STATE>(F, N, nb); });
    else load_incoming<Q, T, true, STATE>(F, N, nb, f);
    if (out) static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; out[(size_t)i * N + idx] = f[i]; });
    if (p) {
        Moments<Q, T, false> m;
        m.compute(f);
        p[idx] = m.m0 * (rho_L + C[idx] * drho) * T(1.0 / 3.0);
    }
}

// Import: POST convention -> ST_SWAP storage (local permutation), or incoming convention -> ST_POST
// storage (Fs_i(y) = f_i(y+e_i), or f_ibar(y) if y+e_i lies beyond a wall).  The other two cases
// (POST -> ST_POST, incoming -> ST_IN) are plain copies.
template <typename T, int Q, bool POST>
__global__ void import_kernel(const T* __restrict__ in, T* F, Geom g, size_t N)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z * blockDim.z + threadIdx.z;
    if (x >= g.nx || y >= g.ny || z >= g.nz) return;
    Nbr nb;
    nb.setup<true>(g, x, y, z);
    const int idx = nb.at<0, 0, 0>();
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        using L = Lat<Q>;
        constexpr int ex = L::ex(i), ey = L::ey(i), ez = L::ez(i);
        if constexpr (POST) {
            F[(size_t)L::opp(i) * N + idx] = in[(size_t)i * N + idx];
        } else {
            const T v = nb.template beyond<ex, ey, ez, true>() ? in[(size_t)L::opp(i) * N + idx]
                                                               : in[(size_t)i * N + nb.template at<ex, ey, ez>()];
            F[(size_t)i * N + idx] = v;
        }
    });
}

// deterministic two-pass sum: fixed grid, fixed per-thread order, shuffle tree, fixed final order
constexpr int RED_BLOCKS = 592, RED_THREADS = 256;   // 4 CTAs per SM on 148 SMs

__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double warp_part[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) warp_part[wid] = v;
    __syncthreads();
    v = (threadIdx.x < (blockDim.x >> 5)) ? warp_part[threadIdx.x] : 0.0;
    if (wid == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;
}

template <typename T>
__global__ void __launch_bounds__(RED_THREADS) sum_pass1(const T* __restrict__ C, size_t N, double* part)
{
    double s = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) s += (double)C[i];
    s = block_sum(s);
    if (threadIdx.x == 0) part[blockIdx.x] = s;
}

__global__ void __launch_bounds__(RED_THREADS) sum_pass2(const double* __restrict__ part, int n, double* out)
{
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) s += part[i];
    s = block_sum(s);
    if (threadIdx.x == 0) *out = s;
}

}  // namespace acm

// ==========================================================================================
// Host side: context, dispatch, C ABI
// ==========================================================================================
using namespace acm;

static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

struct acm_ctx {
    int nx, ny, nz, Qh, Qg, precision;
    size_t N, esz;
    double rho_H, rho_L, sigma, xi, M, nu_H, nu_L, grav[3];
    unsigned walls;
    cudaStream_t stream;
    char* ws;
    // carved workspace (byte offsets)
    size_t offH[2], offG[2], offC[2], offU, offStage, offRed;
    int curH, curG, curC;       // which buffer holds the current state
    unsigned options;           // ACM_OPT_*
    int stH, stG;               // storage state of the current H / G buffer (ST_POST | ST_IN | ST_SWAP)
    bool initialised;
    int sticky;                 // ACM_OK or ACM_ECUDA
    dim3 block;
    long long launches;
    // optional per-kernel timing (acm_profile): events recorded around every LB kernel
    bool profiling;
    std::vector<cudaEvent_t> ev;     // per acm_step call: e0 [phase] e1 [hydro] e2 [phase] ...
    std::vector<int> ev_calls;       // number of steps of each recorded acm_step call
};

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

static bool valid_stencil(int q) { return q == 15 || q == 19 || q == 27; }

struct Layout {
    size_t offH[2], offG[2], offC[2], offU, offStage, offRed, total;
};

static bool make_layout(int nx, int ny, int nz, int Qh, int Qg, int precision, unsigned options, Layout* L)
{
    if (options & ~(unsigned)ACM_OPT_ALL) return false;
    const int grids = (options & ACM_OPT_INPLACE) ? 1 : 2;
    if (nx <= 0 || ny <= 0 || nz <= 0 || !valid_stencil(Qh) || !valid_stencil(Qg)) return false;
    if (precision != ACM_F64 && precision != ACM_F32) return false;
    const double cells = (double)nx * ny * nz;
    if (cells >= 2147483648.0) return false;
    const size_t N = (size_t)nx * ny * nz, e = precision == ACM_F64 ? 8 : 4;
    size_t o = 0;
    for (int b = 0; b < grids; ++b) { L->offH[b] = o; o = align256(o + (size_t)Qh * N * e); }
    for (int b = 0; b < grids; ++b) { L->offG[b] = o; o = align256(o + (size_t)Qg * N * e); }
    if (grids == 1) { L->offH[1] = L->offH[0]; L->offG[1] = L->offG[0]; }
    for (int b = 0; b < 2; ++b) { L->offC[b] = o; o = align256(o + N * e); }
    L->offU = o; o = align256(o + 3 * N * e);
    L->offStage = o; o = align256(o + 5 * N * e);
    L->offRed = o; o = align256(o + (RED_BLOCKS + 1) * sizeof(double));
    L->total = o;
    return true;
}

static int check_launch(acm_ctx* c, const char* what)
{
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        c->sticky = ACM_ECUDA;
        return fail(ACM_ECUDA, "%s: %s", what, cudaGetErrorString(e));
    }
    return ACM_OK;
}

static dim3 grid_for(const acm_ctx* c, dim3 b)
{
    return dim3((c->nx + b.x - 1) / b.x, (c->ny + b.y - 1) / b.y, (c->nz + b.z - 1) / b.z);
}

template <typename T> static T* wsp(acm_ctx* c, size_t off) { return reinterpret_cast<T*>(c->ws + off); }

// ---- typed implementations -----------------------------------------------------------------
template <typename T, int QH, int QG>
static int do_init(acm_ctx* c, const T* phi, const T* u)
{
    Geom g{c->nx, c->ny, c->nz, c->walls};
    dim3 b(128, 1, 1), gr = grid_for(c, b);
    T *H = wsp<T>(c, c->offH[0]), *G = wsp<T>(c, c->offG[0]), *C = wsp<T>(c, c->offC[0]), *U = wsp<T>(c, c->offU);
    if (c->options & ACM_OPT_INPLACE) {
        init_kernel<T, QH, QG, true><<<gr, b, 0, c->stream>>>(phi, u, H, G, C, U, g, c->N);
        c->stH = ST_SWAP; c->stG = ST_IN;
    } else {
        init_kernel<T, QH, QG, false><<<gr, b, 0, c->stream>>>(phi, u, H, G, C, U, g, c->N);
        c->stH = c->stG = ST_POST;
    }
    c->curH = c->curG = c->curC = 0;
    return check_launch(c, "init_kernel");
}

// launches K<T, Q, WALLS, STATE> for the runtime (walls, state) pair
#define ACM_LAUNCH_STATE(KERNEL, TT, QQ, walls, state, gr, b, stream, args)                          \
    do {                                                                                              \
        if (walls) {                                                                                  \
            if (state == ST_POST) KERNEL<TT, QQ, true, ST_POST><<<gr, b, 0, stream>>>(args);          \
            else if (state == ST_IN) KERNEL<TT, QQ, true, ST_IN><<<gr, b, 0, stream>>>(args);         \
            else KERNEL<TT, QQ, true, ST_SWAP><<<gr, b, 0, stream>>>(args);                           \
        } else {                                                                                      \
            if (state == ST_POST) KERNEL<TT, QQ, false, ST_POST><<<gr, b, 0, stream>>>(args);         \
            else if (state == ST_IN) KERNEL<TT, QQ, false, ST_IN><<<gr, b, 0, stream>>>(args);        \
            else KERNEL<TT, QQ, false, ST_SWAP><<<gr, b, 0, stream>>>(args);                          \
        }                                                                                             \
    } while (0)

// state of the array after a step that read it in state s
static int next_state(int s) { return s == ST_POST ? ST_POST : (s == ST_IN ? ST_SWAP : ST_IN); }

template <typename T, int QH>
static int launch_phase(acm_ctx* c)
{
    PhaseArgs<T> a;
    a.Hsrc = wsp<T>(c, c->offH[c->curH]); a.Hdst = wsp<T>(c, c->offH[c->curH ^ 1]);
    a.Csrc = wsp<T>(c, c->offC[c->curC]); a.Cdst = wsp<T>(c, c->offC[c->curC ^ 1]);
    a.U = wsp<T>(c, c->offU);
    a.g = Geom{c->nx, c->ny, c->nz, c->walls};
    a.N = c->N;
    const double omega = 1.0 / (3.0 * c->M + 0.5);     // tau_phi = M/c_s^2 (eq. 2), shifted by 1/2
    a.one_minus_omega = (T)(1.0 - omega);
    a.inv_xi = (T)(1.0 / c->xi);
    dim3 b = c->block, gr = grid_for(c, b);
    ACM_LAUNCH_STATE(phase_kernel, T, QH, c->walls, c->stH, gr, b, c->stream, a);
    c->curH ^= 1; c->curC ^= 1;
    c->stH = next_state(c->stH);
    return check_launch(c, "phase_kernel");
}

template <typename T, int QG>
static int launch_hydro(acm_ctx* c)
{
    HydroArgs<T> a;
    a.Gsrc = wsp<T>(c, c->offG[c->curG]); a.Gdst = wsp<T>(c, c->offG[c->curG ^ 1]);
    a.C = wsp<T>(c, c->offC[c->curC]);
    a.U = wsp<T>(c, c->offU);
    a.g = Geom{c->nx, c->ny, c->nz, c->walls};
    a.N = c->N;
    a.rho_L = (T)c->rho_L; a.drho = (T)(c->rho_H - c->rho_L);
    a.tau_L = (T)(3.0 * c->nu_L); a.dtau = (T)(3.0 * c->nu_H - 3.0 * c->nu_L);
    a.beta4 = (T)(4.0 * 12.0 * c->sigma / c->xi); a.kappa = (T)(1.5 * c->sigma * c->xi);
    a.gx = (T)c->grav[0]; a.gy = (T)c->grav[1]; a.gz = (T)c->grav[2];
    dim3 b = c->block, gr = grid_for(c, b);
    ACM_LAUNCH_STATE(hydro_kernel, T, QG, c->walls, c->stG, gr, b, c->stream, a);
    c->curG ^= 1;
    c->stG = next_state(c->stG);
    return check_launch(c, "hydro_kernel");
}

// export of H (post-collision convention) or G (incoming convention, optionally p) from the current state
template <typename T, int Q, bool POST>
static int do_export(acm_ctx* c, const T* F, int state, T* out, T* p)
{
    Geom g{c->nx, c->ny, c->nz, c->walls};
    dim3 b(128, 1, 1), gr = grid_for(c, b);
    const T* C = wsp<T>(c, c->offC[c->curC]);
    const T rl = (T)c->rho_L, dr = (T)(c->rho_H - c->rho_L);
    if (state == ST_POST) export_kernel<T, Q, ST_POST, POST><<<gr, b, 0, c->stream>>>(F, C, out, p, g, c->N, rl, dr);
    else if (state == ST_IN) export_kernel<T, Q, ST_IN, POST><<<gr, b, 0, c->stream>>>(F, C, out, p, g, c->N, rl, dr);
    else export_kernel<T, Q, ST_SWAP, POST><<<gr, b, 0, c->stream>>>(F, C, out, p, g, c->N, rl, dr);
    return check_launch(c, "export_kernel");
}

template <typename T, int Q, bool POST>
static int do_import(acm_ctx* c, const T* in, T* F)
{
    Geom g{c->nx, c->ny, c->nz, c->walls};
    dim3 b(128, 1, 1);
    import_kernel<T, Q, POST><<<grid_for(c, b), b, 0, c->stream>>>(in, F, g, c->N);
    return check_launch(c, "import_kernel");
}

// ---- dispatch over (precision, stencils) ---------------------------------------------------
#define ACM_DISPATCH_Q(q, QQ, ...)                                 \
    switch (q) {                                                    \
        case 15: { constexpr int QQ = 15; __VA_ARGS__; } break;     \
        case 19: { constexpr int QQ = 19; __VA_ARGS__; } break;     \
        default: { constexpr int QQ = 27; __VA_ARGS__; } break;     \
    }

template <typename T>
static int init_t(acm_ctx* c, const void* phi, const void* u)
{
    int rc = ACM_OK;
    ACM_DISPATCH_Q(c->Qh, QH, ACM_DISPATCH_Q(c->Qg, QG, rc = (do_init<T, QH, QG>(c, (const T*)phi, (const T*)u))));
    return rc;
}

static void prof_mark(acm_ctx* c)
{
    if (!c->profiling) return;
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    cudaEventRecord(e, c->stream);
    c->ev.push_back(e);
}

template <typename T>
static int step_t(acm_ctx* c, int n)
{
    if (c->profiling && n > 0) { c->ev_calls.push_back(n); prof_mark(c); }
    for (int t = 0; t < n; ++t) {
        int rc = ACM_OK;
        ACM_DISPATCH_Q(c->Qh, QH, rc = launch_phase<T, QH>(c));
        if (rc) return rc;
        prof_mark(c);
        ACM_DISPATCH_Q(c->Qg, QG, rc = launch_hydro<T, QG>(c));
        if (rc) return rc;
        prof_mark(c);
    }
    return ACM_OK;
}

template <typename T>
static int export_g_t(acm_ctx* c, void* g, void* p)
{
    int rc = ACM_OK;
    ACM_DISPATCH_Q(c->Qg, QG, rc = (do_export<T, QG, false>(c, wsp<T>(c, c->offG[c->curG]), c->stG, (T*)g, (T*)p)));
    return rc;
}

template <typename T>
static int export_h_t(acm_ctx* c, void* h)
{
    int rc = ACM_OK;
    ACM_DISPATCH_Q(c->Qh, QH, rc = (do_export<T, QH, true>(c, wsp<T>(c, c->offH[c->curH]), c->stH, (T*)h, (T*)nullptr)));
    return rc;
}

template <typename T>
static int import_g_t(acm_ctx* c, const void* g)      // incoming convention -> ST_POST storage
{
    int rc = ACM_OK;
    ACM_DISPATCH_Q(c->Qg, QG, rc = (do_import<T, QG, false>(c, (const T*)g, wsp<T>(c, c->offG[c->curG]))));
    return rc;
}

template <typename T>
static int import_h_t(acm_ctx* c, const void* h)      // post-collision convention -> ST_SWAP storage
{
    int rc = ACM_OK;
    ACM_DISPATCH_Q(c->Qh, QH, rc = (do_import<T, QH, true>(c, (const T*)h, wsp<T>(c, c->offH[c->curH]))));
    return rc;
}

static int copy_async(acm_ctx* c, void* dst, const void* src, size_t bytes, cudaMemcpyKind kind, const char* what)
{
    cudaError_t e = cudaMemcpyAsync(dst, src, bytes, kind, c->stream);
    if (e != cudaSuccess) {
        c->sticky = ACM_ECUDA;
        return fail(ACM_ECUDA, "%s: %s", what, cudaGetErrorString(e));
    }
    return ACM_OK;
}

#define ACM_CHECK_CTX(c)                                                          \
    if (!(c)) return fail(ACM_EINVAL, "%s: NULL context", __func__);              \
    if ((c)->sticky) return fail(ACM_ECUDA, "%s: context has a sticky CUDA error", __func__)

// ---- C ABI ----------------------------------------------------------------------------------
extern "C" {

const char* acm_last_error(void) { return g_err; }

size_t acm_workspace_bytes(int nx, int ny, int nz, int stencil_phase, int stencil_hydro, int precision)
{
    return acm_workspace_bytes_opt(nx, ny, nz, stencil_phase, stencil_hydro, precision, 0u);
}

size_t acm_workspace_bytes_opt(int nx, int ny, int nz, int stencil_phase, int stencil_hydro, int precision, unsigned options)
{
    Layout L;
    return make_layout(nx, ny, nz, stencil_phase, stencil_hydro, precision, options, &L) ? L.total : 0;
}

int acm_create(acm_ctx** out, int nx, int ny, int nz, int stencil_phase, int stencil_hydro, double rho_H, double rho_L,
               double sigma, double xi, double M, double nu_H, double nu_L, const double gravity[3], unsigned wall_flags,
               int precision, void* workspace, void* cuda_stream)
{
    return acm_create_opt(out, nx, ny, nz, stencil_phase, stencil_hydro, rho_H, rho_L, sigma, xi, M, nu_H, nu_L, gravity,
                          wall_flags, precision, 0u, workspace, cuda_stream);
}

int acm_create_opt(acm_ctx** out, int nx, int ny, int nz, int stencil_phase, int stencil_hydro, double rho_H, double rho_L,
                   double sigma, double xi, double M, double nu_H, double nu_L, const double gravity[3], unsigned wall_flags,
                   int precision, unsigned options, void* workspace, void* cuda_stream)
{
    if (!out) return fail(ACM_EINVAL, "acm_create: out is NULL");
    *out = nullptr;
    Layout L;
    if (!make_layout(nx, ny, nz, stencil_phase, stencil_hydro, precision, options, &L))
        return fail(ACM_EINVAL, "acm_create: invalid size (%d,%d,%d), stencils (%d,%d), precision %d or options %u", nx, ny, nz,
                    stencil_phase, stencil_hydro, precision, options);
    if (!(rho_L > 0.0) || !(rho_H >= rho_L)) return fail(ACM_EINVAL, "acm_create: need rho_H >= rho_L > 0");
    if (!(xi > 0.0)) return fail(ACM_EINVAL, "acm_create: need xi > 0");
    if (!(sigma >= 0.0)) return fail(ACM_EINVAL, "acm_create: need sigma >= 0");
    if (!(M > 0.0) || !std::isfinite(M)) return fail(ACM_EINVAL, "acm_create: need mobility M > 0");
    if (!(nu_H > 0.0) || !(nu_L > 0.0)) return fail(ACM_EINVAL, "acm_create: need nu_H, nu_L > 0");
    if (wall_flags & ~7u) return fail(ACM_EINVAL, "acm_create: unknown wall flag");
    if (!workspace) return fail(ACM_EINVAL, "acm_create: workspace is NULL");
    if ((uintptr_t)workspace & 255) return fail(ACM_EINVAL, "acm_create: workspace must be 256-byte aligned");
    acm_ctx* c = new (std::nothrow) acm_ctx();
    if (!c) return fail(ACM_EINVAL, "acm_create: out of host memory");
    c->nx = nx; c->ny = ny; c->nz = nz; c->Qh = stencil_phase; c->Qg = stencil_hydro; c->precision = precision;
    c->N = (size_t)nx * ny * nz; c->esz = precision == ACM_F64 ? 8 : 4;
    c->rho_H = rho_H; c->rho_L = rho_L; c->sigma = sigma; c->xi = xi; c->M = M; c->nu_H = nu_H; c->nu_L = nu_L;
    for (int a = 0; a < 3; ++a) c->grav[a] = gravity ? gravity[a] : 0.0;
    c->walls = wall_flags;
    c->stream = (cudaStream_t)cuda_stream;
    c->ws = (char*)workspace;
    for (int b = 0; b < 2; ++b) { c->offH[b] = L.offH[b]; c->offG[b] = L.offG[b]; c->offC[b] = L.offC[b]; }
    c->offU = L.offU; c->offStage = L.offStage; c->offRed = L.offRed;
    c->curH = c->curG = c->curC = 0;
    c->options = options;
    c->stH = c->stG = ST_POST;
    c->initialised = false;
    c->sticky = ACM_OK;
    c->block = dim3(128, 1, 1);
    c->launches = 0;
    c->profiling = false;
    *out = c;
    return ACM_OK;
}

static void prof_clear(acm_ctx* c)
{
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    c->ev.clear();
    c->ev_calls.clear();
}

void acm_destroy(acm_ctx* c)
{
    if (!c) return;
    prof_clear(c);
    delete c;
}

int acm_profile(acm_ctx* c, int enable)
{
    ACM_CHECK_CTX(c);
    prof_clear(c);
    c->profiling = enable != 0;
    return ACM_OK;
}

int acm_profile_read(acm_ctx* c, double* phase_ms, double* hydro_ms, long long* steps)
{
    ACM_CHECK_CTX(c);
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "acm_profile_read: %s", cudaGetErrorString(e)); }
    double ph = 0.0, hy = 0.0;
    long long ns = 0;
    size_t k = 0;
    for (int n : c->ev_calls) {
        if (k + 2 * (size_t)n + 1 > c->ev.size()) break;
        for (int t = 0; t < n; ++t) {
            float a = 0.f, b = 0.f;
            cudaEventElapsedTime(&a, c->ev[k + 2 * t], c->ev[k + 2 * t + 1]);
            cudaEventElapsedTime(&b, c->ev[k + 2 * t + 1], c->ev[k + 2 * t + 2]);
            ph += a; hy += b;
        }
        ns += n;
        k += 2 * (size_t)n + 1;
    }
    if (phase_ms) *phase_ms = ph;
    if (hydro_ms) *hydro_ms = hy;
    if (steps) *steps = ns;
    prof_clear(c);
    return ACM_OK;
}

int acm_set_block(acm_ctx* c, int bx, int by, int bz)
{
    ACM_CHECK_CTX(c);
    if (bx < 1 || by < 1 || bz < 1 || (long long)bx * by * bz > 256 || bz > 64)
        return fail(ACM_EINVAL, "acm_set_block: need 1 <= bx*by*bz <= 256");
    c->block = dim3(bx, by, bz);
    return ACM_OK;
}

long long acm_launch_count(const acm_ctx* c) { return c ? c->launches : 0; }

int acm_init(acm_ctx* c, const void* phi, const void* u)
{
    ACM_CHECK_CTX(c);
    if (!phi || !u) return fail(ACM_EINVAL, "acm_init: phi and u are required");
    int rc = c->precision == ACM_F64 ? init_t<double>(c, phi, u) : init_t<float>(c, phi, u);
    if (rc == ACM_OK) c->initialised = true;
    return rc;
}

int acm_step(acm_ctx* c, int n)
{
    ACM_CHECK_CTX(c);
    if (n < 0) return fail(ACM_EINVAL, "acm_step: n must be >= 0");
    if (!c->initialised) return fail(ACM_ESTATE, "acm_step: call acm_init first");
    return c->precision == ACM_F64 ? step_t<double>(c, n) : step_t<float>(c, n);
}

int acm_fields(acm_ctx* c, void* phi, void* u, void* p)
{
    ACM_CHECK_CTX(c);
    if (!c->initialised) return fail(ACM_ESTATE, "acm_fields: call acm_init first");
    int rc = ACM_OK;
    if (phi) rc = copy_async(c, phi, c->ws + c->offC[c->curC], c->N * c->esz, cudaMemcpyDeviceToDevice, "acm_fields(phi)");
    if (!rc && u) rc = copy_async(c, u, c->ws + c->offU, 3 * c->N * c->esz, cudaMemcpyDeviceToDevice, "acm_fields(u)");
    if (!rc && p) rc = c->precision == ACM_F64 ? export_g_t<double>(c, nullptr, p) : export_g_t<float>(c, nullptr, p);
    return rc;
}

int acm_phi_mass(acm_ctx* c, double* total_host)
{
    ACM_CHECK_CTX(c);
    if (!total_host) return fail(ACM_EINVAL, "acm_phi_mass: total_host is NULL");
    if (!c->initialised) return fail(ACM_ESTATE, "acm_phi_mass: call acm_init first");
    double* part = wsp<double>(c, c->offRed);
    if (c->precision == ACM_F64)
        sum_pass1<double><<<RED_BLOCKS, RED_THREADS, 0, c->stream>>>(wsp<double>(c, c->offC[c->curC]), c->N, part);
    else
        sum_pass1<float><<<RED_BLOCKS, RED_THREADS, 0, c->stream>>>(wsp<float>(c, c->offC[c->curC]), c->N, part);
    int rc = check_launch(c, "sum_pass1");
    if (rc) return rc;
    sum_pass2<<<1, RED_THREADS, 0, c->stream>>>(part, RED_BLOCKS, part + RED_BLOCKS);
    rc = check_launch(c, "sum_pass2");
    if (rc) return rc;
    rc = copy_async(c, total_host, part + RED_BLOCKS, sizeof(double), cudaMemcpyDeviceToHost, "acm_phi_mass");
    if (rc) return rc;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "acm_phi_mass: %s", cudaGetErrorString(e)); }
    if (!std::isfinite(*total_host)) return fail(ACM_EUNSTABLE, "acm_phi_mass: sum(phi) is not finite");
    return ACM_OK;
}

int acm_get_pdfs(acm_ctx* c, void* h, void* g)
{
    ACM_CHECK_CTX(c);
    if (!c->initialised) return fail(ACM_ESTATE, "acm_get_pdfs: call acm_init first");
    int rc = ACM_OK;
    if (h) rc = c->precision == ACM_F64 ? export_h_t<double>(c, h) : export_h_t<float>(c, h);
    if (!rc && g) rc = c->precision == ACM_F64 ? export_g_t<double>(c, g, nullptr) : export_g_t<float>(c, g, nullptr);
    return rc;
}

int acm_set_pdfs(acm_ctx* c, const void* h, const void* g)
{
    ACM_CHECK_CTX(c);
    if (!c->initialised) return fail(ACM_ESTATE, "acm_set_pdfs: call acm_init first");
    int rc = ACM_OK;
    const bool inplace = (c->options & ACM_OPT_INPLACE) != 0;
    if (h) {
        // post-collision convention: two-grid stores it as is (ST_POST); in place as ST_SWAP
        if (inplace) { rc = c->precision == ACM_F64 ? import_h_t<double>(c, h) : import_h_t<float>(c, h); c->stH = ST_SWAP; }
        else rc = copy_async(c, c->ws + c->offH[c->curH], h, (size_t)c->Qh * c->N * c->esz, cudaMemcpyDeviceToDevice, "acm_set_pdfs(h)");
    }
    if (!rc && g) {
        // incoming convention: in place stores it as is (ST_IN); two-grid pre-shifts it into ST_POST
        if (inplace) { rc = copy_async(c, c->ws + c->offG[c->curG], g, (size_t)c->Qg * c->N * c->esz, cudaMemcpyDeviceToDevice, "acm_set_pdfs(g)"); c->stG = ST_IN; }
        else rc = c->precision == ACM_F64 ? import_g_t<double>(c, g) : import_g_t<float>(c, g);
    }
    return rc;
}

int acm_run_host(acm_ctx* c, const void* phi_host, const void* u_host, int n, void* phi_out_host, void* u_out_host,
                 void* p_out_host)
{
    ACM_CHECK_CTX(c);
    if (!phi_host || !u_host) return fail(ACM_EINVAL, "acm_run_host: phi_host and u_host are required");
    if (n < 0) return fail(ACM_EINVAL, "acm_run_host: n must be >= 0");
    const size_t fb = c->N * c->esz;
    char* st = c->ws + c->offStage;
    int rc = copy_async(c, st, phi_host, fb, cudaMemcpyHostToDevice, "acm_run_host(h2d phi)");
    if (!rc) rc = copy_async(c, st + fb, u_host, 3 * fb, cudaMemcpyHostToDevice, "acm_run_host(h2d u)");
    if (!rc) rc = acm_init(c, st, st + fb);
    if (!rc) rc = acm_step(c, n);
    if (!rc && p_out_host) rc = acm_fields(c, nullptr, nullptr, st + 4 * fb);
    if (!rc && phi_out_host) rc = copy_async(c, phi_out_host, c->ws + c->offC[c->curC], fb, cudaMemcpyDeviceToHost, "acm_run_host(d2h phi)");
    if (!rc && u_out_host) rc = copy_async(c, u_out_host, c->ws + c->offU, 3 * fb, cudaMemcpyDeviceToHost, "acm_run_host(d2h u)");
    if (!rc && p_out_host) rc = copy_async(c, p_out_host, st + 4 * fb, fb, cudaMemcpyDeviceToHost, "acm_run_host(d2h p)");
    if (rc) return rc;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "acm_run_host: %s", cudaGetErrorString(e)); }
    return ACM_OK;
}

}  // extern "C"
