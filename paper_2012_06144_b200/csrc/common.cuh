// common.cuh -- device building blocks shared by the kernel translation units of libacm:
// geometry / neighbour indexing, the storage states of a population array and the streaming they
// imply, the isotropic finite differences of phi, and the argument blocks of the two LB kernels.
// See DESIGN.md for the data layout.  Shares no code with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>

#include "../../include/acm.h"
#include "lattice.cuh"

namespace acm {

// ------------------------------------------------------------------------------------------
// geometry: neighbour indexing with periodic wrap, wall flags for half-way bounce-back
// ------------------------------------------------------------------------------------------
// Internal wall bits: ACM_WALL_X, ACM_WALL_Y as in the ABI; the z walls are kept per face because a
// slab of a z-decomposed domain (acm_create_slab) has a wall on at most one of its faces.
enum { WALL_ZLO = 4, WALL_ZHI = 8 };

struct Geom {
    int nx, ny, nz;  // allocated planes: nz includes the two ghost planes of a slab
    unsigned walls;  // ACM_WALL_X | ACM_WALL_Y | WALL_ZLO | WALL_ZHI
    int linear;      // 1: the launch is 1-D over all cells (rows not a multiple of the block: no idle tail threads)
    int zlo, zhi;    // planes [zlo, zhi) are the cells this context owns ([0, nz) without ghost planes)
    int zghost;      // 1: planes zlo-1 and zhi hold the neighbour slabs' boundary planes (no periodic wrap in z)
    int lz0, lz1;    // planes [lz0, lz1) are covered by this launch (inner / outer split of a slab)
};

// cell of the calling thread: 3-D launch (block tiles of x-rows) or linear launch over the cells of
// the planes [lz0, lz1)
__device__ __forceinline__ bool cell_of_thread(const Geom& g, int& x, int& y, int& z)
{
    if (g.linear) {
        const unsigned id = blockIdx.x * blockDim.x + threadIdx.x;
        if (id >= (unsigned)(g.nx * g.ny * (g.lz1 - g.lz0))) return false;
        const unsigned t = id / (unsigned)g.nx;
        x = (int)(id - t * (unsigned)g.nx);
        const unsigned zr = t / (unsigned)g.ny;
        y = (int)(t - zr * (unsigned)g.ny);
        z = g.lz0 + (int)zr;
        return true;
    }
    x = blockIdx.x * blockDim.x + threadIdx.x;
    y = blockIdx.y * blockDim.y + threadIdx.y;
    z = g.lz0 + blockIdx.z * blockDim.z + threadIdx.z;
    return x < g.nx && y < g.ny && z < g.lz1;
}

// Per-cell neighbourhood: coordinates of x-1, x, x+1 (periodic wrap; clamped at a wall, which is
// the mirror ghost phi(x,-1,z) = phi(x,0,z) of the FD stencils) and "beyond a wall" flags.
struct Nbr {
    // unsigned: cell indices are < 2^31 and a zero-extended index costs one wide multiply-add per address
    unsigned xs[3];        // x-1, x, x+1
    unsigned row[3][3];    // [dz+1][dy+1] -> (z'*ny + y')*nx
    bool wxm, wxp, wym, wyp, wzm, wzp;   // the cell at x-1 / x+1 / ... lies beyond a wall
    bool peer_lo, peer_hi;               // slab: the plane z-1 / z+1 belongs to the low / high neighbour slab

    template <bool WALLS>
    __device__ __forceinline__ void setup(const Geom& g, int x, int y, int z)
    {
        wxm = wxp = wym = wyp = wzm = wzp = false;
        int xm = x - 1, xp = x + 1, ym = y - 1, yp = y + 1, zm = z - 1, zp = z + 1;
        if (xm < 0) { if (WALLS && (g.walls & ACM_WALL_X)) { wxm = true; xm = 0; } else xm = g.nx - 1; }
        if (xp >= g.nx) { if (WALLS && (g.walls & ACM_WALL_X)) { wxp = true; xp = g.nx - 1; } else xp = 0; }
        if (ym < 0) { if (WALLS && (g.walls & ACM_WALL_Y)) { wym = true; ym = 0; } else ym = g.ny - 1; }
        if (yp >= g.ny) { if (WALLS && (g.walls & ACM_WALL_Y)) { wyp = true; yp = g.ny - 1; } else yp = 0; }
        // z: wall -> clamp; ghost planes -> use them as they are; else periodic wrap inside [zlo, zhi)
        if (zm < g.zlo) { if (WALLS && (g.walls & WALL_ZLO)) { wzm = true; zm = g.zlo; } else if (!g.zghost) zm = g.zhi - 1; }
        if (zp >= g.zhi) { if (WALLS && (g.walls & WALL_ZHI)) { wzp = true; zp = g.zhi - 1; } else if (!g.zghost) zp = g.zlo; }
        peer_lo = g.zghost && z == g.zlo && !wzm;
        peer_hi = g.zghost && z == g.zhi - 1 && !wzp;
        xs[0] = (unsigned)xm; xs[1] = (unsigned)x; xs[2] = (unsigned)xp;
        const int ys[3] = {ym, y, yp}, zs[3] = {zm, z, zp};
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) row[a][b] = (unsigned)((zs[a] * g.ny + ys[b]) * g.nx);
    }
    // index of the cell at offset (dx,dy,dz), each in {-1,0,1}
    template <int DX, int DY, int DZ>
    __device__ __forceinline__ unsigned at() const { return row[DZ + 1][DY + 1] + xs[DX + 1]; }
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

// launch bounds of the two LB kernels (the fp32 translation units raise the minimum blocks per SM)
#ifndef ACM_PHASE_MINB
#define ACM_PHASE_MINB 1
#endif
#ifndef ACM_HYDRO_MINB
#define ACM_HYDRO_MINB 1
#endif
#ifndef ACM_MAXT
#define ACM_MAXT 256
#endif

// population loads/stores: plain ld/st.  Measured on B200 (profiles/r1_variants.md): the streaming hints
// (__ldcs/__stcs, __ldg/__stcg) lose 5 % on the whole step against plain accesses.
template <typename T> __device__ __forceinline__ T ld_stream(const T* p) { return *p; }
template <typename T> __device__ __forceinline__ void st_stream(T* p, T v) { *p = v; }

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

// variants of the phase-field collision (ACM_OPT_PHASE_SRT)
enum { PHASE_MRT = 0, PHASE_SRT = 1 };

// Peer mode of a slab (acm_set_peers): what lies in the planes just outside the owned range is read straight from
// the neighbour slabs' arrays -- device pointers into another context's workspace, on this GPU or mapped from a peer
// GPU over NVLink -- instead of from ghost planes filled by an exchange.  `lo` / `hi` are the neighbours' arrays
// shifted such that this slab's own cell index addresses the right plane (equal slab heights).
template <typename T>
struct Peers {
    const T* lo;
    const T* hi;
};

// incoming populations f_i(x) from an array in state STATE
template <int Q, typename T, bool WALLS, int STATE, bool PEER = false>
__device__ __forceinline__ void load_incoming(const T* F, size_t N, const Nbr& nb, T (&f)[Q], Peers<T> peers = Peers<T>{nullptr, nullptr})
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
            const T* base = F;
            if constexpr (PEER && ez > 0) base = nb.peer_lo ? peers.lo : F;      // pulled from the plane z - 1
            if constexpr (PEER && ez < 0) base = nb.peer_hi ? peers.hi : F;      // pulled from the plane z + 1
            src = base + (size_t)far * N + nb.template at<-ex, -ey, -ez>();
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
template <int Q, typename T, bool LAPLACE, typename Acc>
__device__ __forceinline__ void fd_phi_acc(const Acc& acc, T c0, T& gx, T& gy, T& gz, T& lap)
{
    using L = Lat<Q>;
    T dx[4] = {0, 0, 0, 0}, dy[4] = {0, 0, 0, 0}, dz[4] = {0, 0, 0, 0}, ss[4] = {0, 0, 0, 0};   // per class
    static_for<1, Q, 2>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int ex = L::ex(i), ey = L::ey(i), ez = L::ez(i), c = L::cls(i);
        const T p = acc.template get<ex, ey, ez>();
        const T m = acc.template get<-ex, -ey, -ez>();
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

// the phi stencil reads global memory through L1/L2: ncu shows one DRAM read per phi value; a
// shared-memory tile was measured 2-8 % slower (profiles/r1b_profiles.md) and is not kept
template <typename T, bool PEER = false>
struct PhiGlobal {
    const T* C;
    const Nbr* nb;
    Peers<T> peers;
    template <int DX, int DY, int DZ> __device__ __forceinline__ T get() const
    {
        const T* base = C;
        if constexpr (PEER && DZ < 0) base = nb->peer_lo ? peers.lo : C;
        if constexpr (PEER && DZ > 0) base = nb->peer_hi ? peers.hi : C;
        return __ldg(base + nb->template at<DX, DY, DZ>());
    }
};
template <int Q, typename T, bool LAPLACE>
__device__ __forceinline__ void fd_phi(const T* __restrict__ C, const Nbr& nb, T c0, T& gx, T& gy, T& gz, T& lap)
{
    fd_phi_acc<Q, T, LAPLACE>(PhiGlobal<T>{C, &nb, Peers<T>{nullptr, nullptr}}, c0, gx, gy, gz, lap);
}

template <int Q, typename T, bool LAPLACE>
__device__ __forceinline__ void fd_phi_peer(const T* __restrict__ C, const Nbr& nb, Peers<T> peers, T c0, T& gx, T& gy, T& gz, T& lap)
{
    fd_phi_acc<Q, T, LAPLACE>(PhiGlobal<T, true>{C, &nb, peers}, c0, gx, gy, gz, lap);
}

// ------------------------------------------------------------------------------------------
// argument blocks of the two LB kernels
// ------------------------------------------------------------------------------------------
template <typename T>
struct PhaseArgs {
    const T* Hsrc; T* Hdst;
    const T* Csrc; T* Cdst;
    const T* U;
    Geom g;
    unsigned N;      // cells per population plane (< 2^31): 32 bits keep the plane offsets i*N one wide multiply
    T one_minus_omega, inv_xi;
    T ref;           // fp32 instance: reference phase of the deviation storage (0 or 1); 0 for fp64
    Peers<T> Hpeer, Cpeer;   // peer mode of a slab (else unused)
};

template <typename T>
struct HydroArgs {
    const T* Gsrc; T* Gdst;
    const T* C;      // new phi
    T* U;
    Geom g;
    unsigned N;      // cells per population plane (< 2^31): 32 bits keep the plane offsets i*N one wide multiply
    T rho_L, drho, tau_L, dtau, beta4, kappa, gx, gy, gz;
    T ref;           // as in PhaseArgs; rho_L, tau_L are the values at phi = ref
    int bulk_one;    // variant A26 (ACM_OPT_BULK_ONE): the bulk moment relaxes with 1; read by the HVAR = 1 instances only
    int subiter;     // variant A27 (acm_set_subiter): sweeps of the fixed point of eq. 22, >= 1; HVAR = 1 instances only
    Peers<T> Gpeer, Cpeer;   // peer mode of a slab (else unused)
};

// argument blocks of the kernels in moment representation (ACM_OPT_MOMENTS, moment_impl.cuh)
template <typename T>
struct MomPhaseArgs {
    const T* Msrc; T* Mdst;      // [4][N]: A, b of h*
    const T* Csrc; T* Cdst;      // phi
    const T* Uold;               // velocity the collision that wrote Msrc used (read at the neighbours)
    const T* U;                  // current velocity (read at the cell)
    Geom g;
    unsigned N;
    T one_minus_omega, inv_xi;
};

template <typename T>
struct MomHydroArgs {
    HydroArgs<T> h;              // constants, new phi (h.C), geometry; h.Gsrc / h.Gdst / h.U are not used
    const T* Ksrc; T* Kdst;      // [10][N]: A, b, T of g*
    const T* Uin; T* Uout;       // velocity of the previous step (read at the cell) / of this step
};

}  // namespace acm
