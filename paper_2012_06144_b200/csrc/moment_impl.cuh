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
// to 6 (g) / 8 (h) values of the neighbour instead of one.  Three kernel families, all instances of the same pull /
// collide functions over an accessor: DIRECT (one thread per cell, gather through L1/L2), MARCHING (tile of columns
// marching along z, coefficient planes staged in shared memory) and PUSHING (every source cell of the window expanded once
// into destination-indexed shared-memory arrays).  Measurements and the way there: DESIGN.md 5.10, profiles/r2b_profiles.md.
#include "kernels.h"
#include "lb_math.cuh"

namespace acm {

// Where the coefficients come from.  An accessor names a cell by an index (index<DX,DY,DZ>() = the cell at that
// offset from the calling thread's) and hands out the fields of a cell:
//   hydrodynamic set: k(f, j), f = 0..9: A, bx, by, bz, Txx, Tyy, Tzz, Txy, Txz, Tyz
//   phase-field set:  m(f, j), f = 0..3: A, bx, by, bz;  phi(j);  u(a, j): the velocity the collision that wrote m used
// GlobalK / GlobalM read the arrays in global memory through L1/L2; the tile accessors of the marching kernels
// (below) read the shared-memory window.
template <typename T>
struct GlobalK {
    const T* __restrict__ K;
    size_t N;
    const Nbr* nb;
    template <int DX, int DY, int DZ> __device__ __forceinline__ unsigned index() const { return nb->template at<DX, DY, DZ>(); }
    __device__ __forceinline__ T k(int f, unsigned j) const { return __ldg(K + (size_t)f * N + j); }
};

template <typename T>
struct GlobalM {
    const T* __restrict__ M;
    const T* __restrict__ C;
    const T* __restrict__ Uo;
    size_t N;
    const Nbr* nb;
    template <int DX, int DY, int DZ> __device__ __forceinline__ unsigned index() const { return nb->template at<DX, DY, DZ>(); }
    __device__ __forceinline__ T m(int f, unsigned j) const { return __ldg(M + (size_t)f * N + j); }
    __device__ __forceinline__ T phi(unsigned j) const { return __ldg(C + j); }
    __device__ __forceinline__ T u(int a, unsigned j) const { return __ldg(Uo + (size_t)a * N + j); }
};

// "beyond a wall" flags of a cell (the part of Nbr the pulls need; Nbr itself qualifies too)
struct WallFlags {
    bool wxm, wxp, wym, wyp, wzm, wzp;
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

// index of the cell that delivers population I to the calling cell, and whether the delivery is a bounce-back
// (then the cell itself delivers its own opposite population: same even part, odd part with the other sign)
template <int Q, int I, bool WALLS, bool LOCAL, typename Acc, typename Walls>
__device__ __forceinline__ auto mom_source(const Acc& acc, const Walls& wf, bool& flip)
{
    using L = Lat<Q>;
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I);
    flip = false;
    if constexpr (LOCAL || I == 0) return acc.template index<0, 0, 0>();
    else {
        if constexpr (WALLS) {
            if (wf.template beyond<-ex, -ey, -ez, WALLS>()) { flip = true; return acc.template index<0, 0, 0>(); }
        }
        return acc.template index<-ex, -ey, -ez>();
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

// incoming hydrodynamic population g_I(x) / w_I rebuilt from the coefficients.
// LOCAL: the coefficients are those of the cell's own INCOMING populations (state right after acm_init, whose g is
// defined pre-collision at its cell, A13/A14): no streaming.
template <int Q, int I, typename T, bool WALLS, bool LOCAL, typename Acc, typename Walls>
__device__ __forceinline__ T mom_pull_g(const Acc& acc, const Walls& wf)
{
    using L = Lat<Q>;
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I);
    bool flip;
    const auto j = mom_source<Q, I, WALLS, LOCAL>(acc, wf, flip);
    T E = acc.k(0, j);                                           // A
    if constexpr (ex != 0) E += acc.k(4, j);                     // e e : T, diagonal part
    if constexpr (ey != 0) E += acc.k(5, j);
    if constexpr (ez != 0) E += acc.k(6, j);
    if constexpr (ex * ey != 0) E += T(2 * ex * ey) * acc.k(7, j);
    if constexpr (ex * ez != 0) E += T(2 * ex * ez) * acc.k(8, j);
    if constexpr (ey * ez != 0) E += T(2 * ey * ez) * acc.k(9, j);
    if constexpr (I == 0) return E;
    else {
        T O = T(0);
        bool first = true;
        if constexpr (ex != 0) odd_term<ex>(O, first, acc.k(1, j));
        if constexpr (ey != 0) odd_term<ey>(O, first, acc.k(2, j));
        if constexpr (ez != 0) odd_term<ez>(O, first, acc.k(3, j));
        if constexpr (WALLS) return flip ? E - O : E + O;
        else return E + O;
    }
}

// incoming phase-field population h_I(x) / w_I rebuilt from A, b, phi and the velocity the collision that wrote
// them used:  h*_i = w_i [A + e_i.b + 4.5 phi (e_i.u)^2],  A = phi (1 - 1.5 u^2),  b = 3 phi u + forcing + relaxed part
template <int Q, int I, typename T, bool WALLS, bool LOCAL, typename Acc, typename Walls>
__device__ __forceinline__ T mom_pull_h(const Acc& acc, const Walls& wf)
{
    using L = Lat<Q>;
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I);
    bool flip;
    const auto j = mom_source<Q, I, WALLS, LOCAL>(acc, wf, flip);
    const T A = acc.m(0, j);
    if constexpr (I == 0) return A;
    else {
        T O = T(0), eu = T(0);
        bool fo = true, fu = true;
        if constexpr (ex != 0) { odd_term<ex>(O, fo, acc.m(1, j)); odd_term<ex>(eu, fu, acc.u(0, j)); }
        if constexpr (ey != 0) { odd_term<ey>(O, fo, acc.m(2, j)); odd_term<ey>(eu, fu, acc.u(1, j)); }
        if constexpr (ez != 0) { odd_term<ez>(O, fo, acc.m(3, j)); odd_term<ez>(eu, fu, acc.u(2, j)); }
        const T E = A + T(4.5) * acc.phi(j) * (eu * eu);
        if constexpr (WALLS) return flip ? E - O : E + O;
        else return E + O;
    }
}

// the rest of the two cell updates, shared by the direct and the marching kernels
// phase field: from the pulled populations h, the OLD phi at the cell and its gradient, and u: phi_new and A, b of h*
// (the MRT branch of phase_collide, lb_math.cuh, up to the coefficients)
template <typename T, int Q>
__device__ __forceinline__ void phase_mom_cell(const T (&h)[Q], T c0, T gx, T gy, T gz, T ux, T uy, T uz, T one_minus_omega, T inv_xi,
                                               T& phi, T& A, T& bx, T& by, T& bz)
{
    Moments<Q, T, false> m;
    m.compute(h);
    phi = m.m0;
    const T g2 = gx * gx + gy * gy + gz * gz;
    const T inv = inv_norm_or_zero(g2);
    const T dc = c0 - T(0.5);
    const T theta = (T(1) - T(4) * dc * dc) * inv_xi;
    const T tnx = theta * inv * gx, tny = theta * inv * gy, tnz = theta * inv * gz;
    const T k = T(3) * one_minus_omega;
    const T sixth = T(1.0 / 6.0);
    const T dxm = m.jx - phi * ux + sixth * tnx;
    const T dym = m.jy - phi * uy + sixth * tny;
    const T dzm = m.jz - phi * uz + sixth * tnz;
    const T p3 = T(3) * phi;
    const T usq = T(1.5) * (ux * ux + uy * uy + uz * uz);
    A = phi * (T(1) - usq);
    bx = p3 * ux + T(0.5) * tnx + k * dxm;
    by = p3 * uy + T(0.5) * tny + k * dym;
    bz = p3 * uz + T(0.5) * tnz + k * dzm;
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

    const GlobalM<T> acc{a.Msrc, a.Csrc, a.Uold, N, &nb};
    T h[Q];
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        h[i] = T(Lat<Q>::w(i)) * mom_pull_h<Q, i, T, WALLS, false>(acc, nb);
    });
    const T ux = __ldg(a.U + idx), uy = __ldg(a.U + N + idx), uz = __ldg(a.U + 2 * N + idx);
    const T c0 = __ldg(a.Csrc + idx);
    T gx, gy, gz, lap_unused;
    fd_phi<Q, T, false>(a.Csrc, nb, c0, gx, gy, gz, lap_unused);
    T phi, A, bx, by, bz;
    phase_mom_cell<T, Q>(h, c0, gx, gy, gz, ux, uy, uz, a.one_minus_omega, a.inv_xi, phi, A, bx, by, bz);
    a.Mdst[idx] = A; a.Mdst[N + idx] = bx; a.Mdst[2 * N + idx] = by; a.Mdst[3 * N + idx] = bz;
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

    const GlobalK<T> acc{a.Ksrc, N, &nb};
    T g[Q];
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        g[i] = T(Lat<Q>::w(i)) * mom_pull_g<Q, i, T, WALLS, LOCAL>(acc, nb);
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
// The marching kernels.  The direct kernels above are latency-bound: each thread issues ~110 dependent-free but
// register-limited loads per cell through L1 (ncu: DRAM at half its rate, nothing else saturated).  Here a block owns a
// TX x TY tile of columns and marches along z over `zchunk` planes; the coefficient planes it needs (tile + one-cell
// halo, periodic wrap / wall clamp applied by the loader; phi and -- for the phase-field step -- the velocity staged with
// them) travel global -> shared memory by cp.async into a ring of plane slots.  Phase-field kernel: four slots, plane z+2
// is in flight while plane z is computed from the slots of z-1, z, z+1, one barrier per plane.  Hydrodynamic kernel (eleven
// fields): three slots, so that two blocks fit an SM; plane z+2 is requested after the computation of plane z.  Every
// coefficient is fetched from L2 once per tile (+ halo), the gather runs on shared memory.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)      // bypasses L1: nothing of the stream is held there
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Tile of one field in a plane slot: ROWS rows (tile + one halo row on each side) of PITCH elements; the cell with
// local x sits in column x + 2, so that the interior starts 16-byte aligned: [pad, halo, TX interior, halo, pad].
// A row is copied by LPR lanes: TX/2 aligned 16-byte chunks and the two halo elements.
template <int TX, int TY, int RING_ = 4>
struct MomTile {
    static constexpr int PITCH = TX + 4, ROWS = TY + 2, TILE = PITCH * ROWS, NT = TX * TY;
    static constexpr int LPR = TX / 2 + 2, LANES = LPR * ROWS;
    static constexpr int RING = RING_;                    // plane slots: 4 = the next plane loads under the computation, 3 = after it
    static_assert(TX % 2 == 0 && LANES <= NT, "one copy lane per thread");
};

// coordinate of a halo / tile entry on one axis: periodic wrap or wall clamp (the mirror ghost of the phi stencil);
// entries beyond the far end of a ragged tile are never used, they only need a valid address
__device__ __forceinline__ int tile_coord(int v, int n, bool wall)
{
    if (v < 0) return wall ? 0 : n - 1;
    if (v >= n) return (v == n && !wall) ? 0 : n - 1;
    return v;
}

// what the two marching kernels share: the block's tile, the thread's copy lane, the z range (needs nx even)
template <typename TL>
struct MarchSetup {
    int x, y, zb, ze;
    bool active;         // the thread's column lies inside the grid
    int copy;            // 0: no copy lane, 8 / 16: bytes of the thread's copy per field and plane
    unsigned src, dst;   // its source offset inside a plane, its destination inside a field tile
    unsigned plane;      // nx * ny
    __device__ __forceinline__ void init(const Geom& g, int zchunk)
    {
        const int tid = threadIdx.y * blockDim.x + threadIdx.x;
        const int x0 = blockIdx.x * (TL::PITCH - 4), y0 = blockIdx.y * (TL::ROWS - 2);
        x = x0 + threadIdx.x; y = y0 + threadIdx.y;
        active = x < g.nx && y < g.ny;
        zb = g.lz0 + blockIdx.z * zchunk;
        ze = min(zb + zchunk, g.lz1);
        plane = (unsigned)(g.nx * g.ny);
        copy = 0; src = dst = 0;
        if (tid < TL::LANES) {
            const int r = tid / TL::LPR, l = tid - r * TL::LPR;
            const int gy = tile_coord(y0 + r - 1, g.ny, (g.walls & ACM_WALL_Y) != 0);
            const bool wx = (g.walls & ACM_WALL_X) != 0;
            int gx, col;
            if (l < TL::LPR - 2) {            // chunk of two interior cells; beyond the end of a ragged row only its first element
                gx = x0 + 2 * l; col = 2 * l + 2;      // (the x + 1 neighbour of the last cell) is ever used
                copy = gx + 1 < g.nx ? 16 : 8;
                if (copy == 8) gx = tile_coord(gx, g.nx, wx);
            } else if (l == TL::LPR - 2) { gx = tile_coord(x0 - 1, g.nx, wx); col = 1; copy = 8; }
            else { gx = tile_coord(x0 + TL::PITCH - 4, g.nx, wx); col = TL::PITCH - 2; copy = 8; }
            src = (unsigned)(gy * g.nx + gx);
            dst = (unsigned)(r * TL::PITCH + col);
        }
    }
    // offset of plane zz (zb - 1 <= zz <= ze): periodic wrap inside [zlo, zhi) or wall clamp
    __device__ __forceinline__ size_t zoff(const Geom& g, int zz) const
    {
        int z = zz;
        if (z < g.zlo) z = (g.walls & WALL_ZLO) ? g.zlo : g.zhi - 1;
        else if (z >= g.zhi) z = (g.walls & WALL_ZHI) ? g.zhi - 1 : g.zlo;
        return (size_t)z * plane;
    }
    __device__ __forceinline__ int slot_of(int zz) const { return TL::RING == 4 ? ((zz - zb + 1) & 3) : (zz - zb + 1) % TL::RING; }
    // copies of one plane: for each of NF fields (field f at base[f]) the thread's lane
    template <int NF, typename T>
    __device__ __forceinline__ void load_plane(T* slot, const T* const (&base)[NF], const Geom& g, int zz) const
    {
        if (copy == 0) return;
        const size_t off = zoff(g, zz) + src;
        T* d = slot + dst;
        if (copy == 16) {
#pragma unroll
            for (int f = 0; f < NF; ++f) cp_async16(d + f * TL::TILE, base[f] + off);
        } else {
#pragma unroll
            for (int f = 0; f < NF; ++f) cp_async8(d + f * TL::TILE, base[f] + off);
        }
    }
};

// shared-memory window as an accessor: base[d] = offset of the thread's own entry in the slot of plane z - 1 + d
template <typename T, typename TL>
struct TileK {      // fields of a slot: 0..9 = A, b, T; 10 = phi
    const T* s;
    int base[3];
    template <int DX, int DY, int DZ> __device__ __forceinline__ int index() const { return base[DZ + 1] + DY * TL::PITCH + DX; }
    __device__ __forceinline__ T k(int f, int j) const { return s[j + f * TL::TILE]; }
    __device__ __forceinline__ T phi(int j) const { return s[j + 10 * TL::TILE]; }
    template <int DX, int DY, int DZ> __device__ __forceinline__ T get() const { return phi(index<DX, DY, DZ>()); }   // fd_phi_acc
};

template <typename T, typename TL>
struct TileM {      // fields of a slot: 0..3 = A, b; 4 = phi; 5..7 = u
    const T* s;
    int base[3];
    template <int DX, int DY, int DZ> __device__ __forceinline__ int index() const { return base[DZ + 1] + DY * TL::PITCH + DX; }
    __device__ __forceinline__ T m(int f, int j) const { return s[j + f * TL::TILE]; }
    __device__ __forceinline__ T phi(int j) const { return s[j + 4 * TL::TILE]; }
    __device__ __forceinline__ T u(int a, int j) const { return s[j + (5 + a) * TL::TILE]; }
    template <int DX, int DY, int DZ> __device__ __forceinline__ T get() const { return phi(index<DX, DY, DZ>()); }   // fd_phi_acc
};

template <typename T, int Q, bool WALLS, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 2) phase_mom_march_kernel(const MomPhaseArgs<T> a, int zchunk)
{
    using TL = MomTile<TX, TY>;
    constexpr int NF = 8;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* s = reinterpret_cast<T*>(smem_raw);      // [RING][NF][TILE]
    const Geom& g = a.g;
    const size_t N = a.N;
    MarchSetup<TL> ms;
    ms.init(g, zchunk);
    if (ms.zb >= ms.ze) return;
    const T* const base[NF] = {a.Msrc, a.Msrc + N, a.Msrc + 2 * N, a.Msrc + 3 * N, a.Csrc, a.Uold, a.Uold + N, a.Uold + 2 * N};
    for (int zz = ms.zb - 1; zz <= ms.zb + 1; ++zz)
        ms.load_plane(s + ms.slot_of(zz) * NF * TL::TILE, base, g, zz);
    cp_async_commit();

    const int own = (threadIdx.y + 1) * TL::PITCH + threadIdx.x + 2;
    WallFlags wf;
    wf.wxm = WALLS && (g.walls & ACM_WALL_X) && ms.x == 0; wf.wxp = WALLS && (g.walls & ACM_WALL_X) && ms.x == g.nx - 1;
    wf.wym = WALLS && (g.walls & ACM_WALL_Y) && ms.y == 0; wf.wyp = WALLS && (g.walls & ACM_WALL_Y) && ms.y == g.ny - 1;
    const unsigned col = (unsigned)(ms.y * g.nx + ms.x);
    for (int z = ms.zb; z < ms.ze; ++z) {
        cp_async_wait_all();
        __syncthreads();      // planes z-1 .. z+1 have landed for everyone, and everyone is done with the slot of z-2
        if (z + 2 <= ms.ze) ms.load_plane(s + ms.slot_of(z + 2) * NF * TL::TILE, base, g, z + 2);
        cp_async_commit();
        if (!ms.active) continue;
        wf.wzm = WALLS && (g.walls & WALL_ZLO) && z == g.zlo; wf.wzp = WALLS && (g.walls & WALL_ZHI) && z == g.zhi - 1;
        TileM<T, TL> acc;
        acc.s = s;
#pragma unroll
        for (int d = 0; d < 3; ++d) acc.base[d] = ms.slot_of(z - 1 + d) * NF * TL::TILE + own;
        T h[Q];
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            h[i] = T(Lat<Q>::w(i)) * mom_pull_h<Q, i, T, WALLS, false>(acc, wf);
        });
        const unsigned idx = (unsigned)z * ms.plane + col;
        const T ux = __ldg(a.U + idx), uy = __ldg(a.U + N + idx), uz = __ldg(a.U + 2 * N + idx);
        const T c0 = acc.phi(acc.base[1]);
        T gx, gy, gz, lap_unused;
        fd_phi_acc<Q, T, false>(acc, c0, gx, gy, gz, lap_unused);
        T phi, A, bx, by, bz;
        phase_mom_cell<T, Q>(h, c0, gx, gy, gz, ux, uy, uz, a.one_minus_omega, a.inv_xi, phi, A, bx, by, bz);
        a.Mdst[idx] = A; a.Mdst[N + idx] = bx; a.Mdst[2 * N + idx] = by; a.Mdst[3 * N + idx] = bz;
        a.Cdst[idx] = phi;
    }
}

// (ring of 3 plane slots: two blocks per SM; the next plane is requested after the computation and lands under the other block's)
template <typename T, int Q, bool WALLS, int HVAR, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 2) hydro_mom_march_kernel(const MomHydroArgs<T> a, int zchunk)
{
    constexpr int RING = 3;
    using TL = MomTile<TX, TY, RING>;
    constexpr int NF = 11;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* s = reinterpret_cast<T*>(smem_raw);      // [RING][NF][TILE]
    const Geom& g = a.h.g;
    const size_t N = a.h.N;
    MarchSetup<TL> ms;
    ms.init(g, zchunk);
    if (ms.zb >= ms.ze) return;
    const T* const base[NF] = {a.Ksrc, a.Ksrc + N, a.Ksrc + 2 * N, a.Ksrc + 3 * N, a.Ksrc + 4 * N,
                               a.Ksrc + 5 * N, a.Ksrc + 6 * N, a.Ksrc + 7 * N, a.Ksrc + 8 * N, a.Ksrc + 9 * N, a.h.C};
    for (int zz = ms.zb - 1; zz <= ms.zb + 1; ++zz)
        ms.load_plane(s + ms.slot_of(zz) * NF * TL::TILE, base, g, zz);
    cp_async_commit();

    const int own = (threadIdx.y + 1) * TL::PITCH + threadIdx.x + 2;
    WallFlags wf;
    wf.wxm = WALLS && (g.walls & ACM_WALL_X) && ms.x == 0; wf.wxp = WALLS && (g.walls & ACM_WALL_X) && ms.x == g.nx - 1;
    wf.wym = WALLS && (g.walls & ACM_WALL_Y) && ms.y == 0; wf.wyp = WALLS && (g.walls & ACM_WALL_Y) && ms.y == g.ny - 1;
    const unsigned col = ms.active ? (unsigned)(ms.y * g.nx + ms.x) : 0u;
    for (int z = ms.zb; z < ms.ze; ++z) {
        // the velocity of the previous step (read at the cell only) is requested before the wait for the window
        const unsigned idx = (unsigned)z * ms.plane + col;
        const T uox = __ldg(a.Uin + idx), uoy = __ldg(a.Uin + N + idx), uoz = __ldg(a.Uin + 2 * N + idx);
        cp_async_wait_all();
        __syncthreads();      // planes z-1 .. z+1 have landed for everyone
        if (ms.active) {
            wf.wzm = WALLS && (g.walls & WALL_ZLO) && z == g.zlo; wf.wzp = WALLS && (g.walls & WALL_ZHI) && z == g.zhi - 1;
            TileK<T, TL> acc;
            acc.s = s;
#pragma unroll
            for (int d = 0; d < 3; ++d) acc.base[d] = ms.slot_of(z - 1 + d) * NF * TL::TILE + own;
            T gp[Q];
            static_for<0, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                gp[i] = T(Lat<Q>::w(i)) * mom_pull_g<Q, i, T, WALLS, false>(acc, wf);
            });
            const T c0 = acc.phi(acc.base[1]);
            T gpx, gpy, gpz, lap;
            fd_phi_acc<Q, T, true>(acc, c0, gpx, gpy, gpz, lap);
            Moments<Q, T, true> m;
            m.compute(gp);
            const HydroCell<T> hc = hydro_velocity<T, Q, HVAR>(m, c0, gpx, gpy, gpz, lap, uox, uoy, uoz, a.h);
            a.Uout[idx] = hc.ux; a.Uout[N + idx] = hc.uy; a.Uout[2 * N + idx] = hc.uz;
            const Coeffs<T> k = hydro_coeffs<T, Q, HVAR>(m, hc, a.h);
            T* o = a.Kdst + idx;
            o[0] = k.A; o[N] = k.bx; o[2 * N] = k.by; o[3 * N] = k.bz;
            o[4 * N] = k.Txx; o[5 * N] = k.Tyy; o[6 * N] = k.Tzz; o[7 * N] = k.Txy; o[8 * N] = k.Txz; o[9 * N] = k.Tyz;
        }
        __syncthreads();      // everyone is done with the slot of z-1: the plane z+2 takes it
        if (z + 2 <= ms.ze) ms.load_plane(s + ms.slot_of(z + 2) * NF * TL::TILE, base, g, z + 2);
        cp_async_commit();
    }
}

// ------------------------------------------------------------------------------------------
// The pushing kernels.  The marching kernels above still gather: ~110 shared-memory loads per cell, which is what
// bounds them (ncu: the shared-memory pipe 60-80 % busy, warps stalled on its queue).  Here every SOURCE cell of the
// window is expanded once: its thread reads the cell's coefficients from global memory into registers (coalesced, requested
// one plane ahead), forms all Q populations with the shared even / odd parts of emit_populations and pushes each one into
// a shared-memory array indexed by its DESTINATION cell; a destination then finds its Q incoming populations at its own
// position -- Q conflict-free loads instead of ~5 Q.  A destination plane z is complete when the source planes z-1, z, z+1
// have been expanded, so the arrays are kept per role: the populations with e_z = +1 of three destination planes, those with
// e_z = 0 of two, those with e_z = -1 of one.  The one-cell halo of the tile is expanded by the first 2 TX + 2 TY + 4 threads
// (only what lands inside the tile is stored).  Bounce-back is applied on the destination side: a cell next to a wall
// rebuilds the populations it cannot receive from its own coefficients.  phi (one field) is staged as in the marching kernels.
// ------------------------------------------------------------------------------------------
// a load the compiler keeps where it is written (the requests of the pushing kernels are placed a phase ahead of their use)
__device__ __forceinline__ double ld_here(const double* p)
{
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float ld_here(const float* p)
{
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}


// mbarrier of a block (shared memory): every thread arrives once per phase, anyone may wait for a phase to complete
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}

template <int Q>
struct PushRoles {
    __host__ __device__ static constexpr int count(int ez) { int n = 0; for (int i = 0; i < Q; ++i) n += Lat<Q>::ez(i) == ez; return n; }
    // position of population I among those with the same e_z
    __host__ __device__ static constexpr int index(int I) { int n = 0; for (int i = 0; i < I; ++i) n += Lat<Q>::ez(i) == Lat<Q>::ez(I); return n; }
    static constexpr int NU = count(1), NM = count(0), ND = count(-1);
};

// accessor that always names the calling cell (bounce-back from its own coefficients)
template <typename T>
struct OwnK {
    const T* __restrict__ K;
    size_t N;
    unsigned idx;
    template <int DX, int DY, int DZ> __device__ __forceinline__ unsigned index() const { return idx; }
    __device__ __forceinline__ T k(int f, unsigned j) const { return __ldg(K + (size_t)f * N + j); }
};

// phi window of the pushing kernels as an accessor for fd_phi_acc
template <typename T, typename TL>
struct TilePhi {
    const T* s;
    int base[3];
    template <int DX, int DY, int DZ> __device__ __forceinline__ T get() const { return s[base[DZ + 1] + DY * TL::PITCH + DX]; }
};

// the source entries of a thread: its own column and, for the first HALO threads, one entry of the ring around the tile
template <int TX, int TY>
struct PushSources {
    // the ring around the tile, one entry per thread: the first TX threads the row below (kind 1), the next TX the row above
    // (2), then the two columns (3, 4) and the corners (5); 0 = none.  The kind is uniform over a warp, except in the one
    // warp that takes the columns and the corners.
    static_assert(TX % 32 == 0 && 2 * TY + 4 <= 32 && 2 * TX + 32 <= TX * TY, "halo assignment by warps");
    int hx, hy;                  // local coordinates of the halo entry
    int kind;
    unsigned own_src, halo_src;  // offsets inside a plane (periodic wrap / wall clamp; a clamped entry pushes values nobody keeps)
    __device__ __forceinline__ void init(const Geom& g)
    {
        const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
        const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
        const bool wx = (g.walls & ACM_WALL_X) != 0, wy = (g.walls & ACM_WALL_Y) != 0;
        own_src = (unsigned)(tile_coord(y0 + ty, g.ny, wy) * g.nx + tile_coord(x0 + tx, g.nx, wx));
        kind = 0; hx = hy = 0;
        if (tid < TX) { hx = tid; hy = -1; kind = 1; }
        else if (tid < 2 * TX) { hx = tid - TX; hy = TY; kind = 2; }
        else if (tid < 2 * TX + TY) { hx = -1; hy = tid - 2 * TX; kind = 3; }
        else if (tid < 2 * TX + 2 * TY) { hx = TX; hy = tid - 2 * TX - TY; kind = 4; }
        else if (tid < 2 * TX + 2 * TY + 4) { const int c = tid - 2 * TX - 2 * TY; hx = (c & 1) ? TX : -1; hy = (c & 2) ? TY : -1; kind = 5; }
        halo_src = (unsigned)(tile_coord(y0 + hy, g.ny, wy) * g.nx + tile_coord(x0 + hx, g.nx, wx));
    }
};

// role arrays of the pushed populations in shared memory
template <typename T, int Q, int TX, int TY>
struct PushBuffers {
    using R = PushRoles<Q>;
    static constexpr int NT = TX * TY;
    static constexpr int DOUBLES = (3 * R::NU + 2 * R::NM + R::ND) * NT;
    T *up, *mid, *dn;
    int zb, ze;
    __device__ __forceinline__ void init(T* s, int zb_, int ze_) { up = s; mid = up + 3 * R::NU * NT; dn = mid + 2 * R::NM * NT; zb = zb_; ze = ze_; }
    __device__ __forceinline__ T* up_of(int k) const { return up + ((k - zb) % 3) * R::NU * NT; }
    __device__ __forceinline__ T* mid_of(int k) const { return mid + ((k - zb) & 1) * R::NM * NT; }
    // bit i: population i of the source entry (sx, sy) lands inside the tile (constant along the march)
    __device__ __forceinline__ static unsigned inside_mask(int sx, int sy)
    {
        unsigned m = 0;
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const int dx = sx + Lat<Q>::ex(i), dy = sy + Lat<Q>::ey(i);
            if ((unsigned)dx < (unsigned)TX && (unsigned)dy < (unsigned)TY) m |= 1u << i;
        });
        return m;
    }
    __host__ __device__ static constexpr unsigned role_bits(int ez)
    {
        unsigned m = 0;
        for (int i = 0; i < Q; ++i) if (Lat<Q>::ez(i) == ez) m |= 1u << i;
        return m;
    }
    // push the populations w_i [A + e_i.b + e_i e_i : T] of the thread's own source entry (position `own`, mask of the
    // populations that land inside the tile) of plane p to their destinations: own + a compile-time offset
    __device__ __forceinline__ void push(int p, int own, unsigned inside, T A, T bx, T by, T bz, T Txx, T Tyy, T Tzz, T Txy, T Txz, T Tyz) const
    {
        const bool okU = p + 1 >= zb && p + 1 < ze, okM = p >= zb && p < ze, okD = p - 1 >= zb && p - 1 < ze;
        const unsigned live = inside & ((okU ? role_bits(1) : 0u) | (okM ? role_bits(0) : 0u) | (okD ? role_bits(-1) : 0u));
        T* const bu = up_of(p + 1) + own;
        T* const bm = mid_of(p) + own;
        T* const bd = dn + own;
        emit_populations<Q, T>(A, bx, by, bz, Txx, Tyy, Tzz, Txy, Txz, Tyz, [&](auto ic, T v) {
            constexpr int i = decltype(ic)::value;
            constexpr int ex = Lat<Q>::ex(i), ey = Lat<Q>::ey(i), ez = Lat<Q>::ez(i), ri = R::index(i);
            constexpr int o = ri * NT + ey * TX + ex;
            if (live & (1u << i)) {
                if constexpr (ez > 0) bu[o] = v;
                else if constexpr (ez == 0) bm[o] = v;
                else bd[o] = v;
            }
        });
    }
    // the same for an entry of the ring around the tile: only the populations that can land inside are formed
    // (RX / RY != 0: only those with e_x = RX / e_y = RY)
    template <int RX, int RY>
    __device__ __forceinline__ void push_from_halo(int p, int sx, int sy, const T (&k)[10]) const
    {
        const bool okU = p + 1 >= zb && p + 1 < ze, okM = p >= zb && p < ze, okD = p - 1 >= zb && p - 1 < ze;
        T* const bu = up_of(p + 1);
        T* const bm = mid_of(p);
        static_for<1, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            constexpr int ex = Lat<Q>::ex(i), ey = Lat<Q>::ey(i), ez = Lat<Q>::ez(i), ri = R::index(i);
            if constexpr ((RX == 0 || ex == RX) && (RY == 0 || ey == RY)) {
                const int dx = sx + ex, dy = sy + ey;
                if ((unsigned)dx < (unsigned)TX && (unsigned)dy < (unsigned)TY) {
                    T E = k[0], O = T(0);
                    bool first = true;
                    if constexpr (ex != 0) { E += k[4]; odd_term<ex>(O, first, k[1]); }
                    if constexpr (ey != 0) { E += k[5]; odd_term<ey>(O, first, k[2]); }
                    if constexpr (ez != 0) { E += k[6]; odd_term<ez>(O, first, k[3]); }
                    if constexpr (ex * ey != 0) E += T(2 * ex * ey) * k[7];
                    if constexpr (ex * ez != 0) E += T(2 * ex * ez) * k[8];
                    if constexpr (ey * ez != 0) E += T(2 * ey * ez) * k[9];
                    const T v = T(Lat<Q>::w(i)) * (E + O);
                    const int o = ri * NT + dy * TX + dx;
                    if constexpr (ez > 0) { if (okU) bu[o] = v; }
                    else if constexpr (ez == 0) { if (okM) bm[o] = v; }
                    else { if (okD) dn[o] = v; }
                }
            }
        });
    }
    // incoming population I of the destination cell at position `own` (= ty * TX + tx) of plane z
    template <int I>
    __device__ __forceinline__ T pull(int z, int own) const
    {
        constexpr int ez = Lat<Q>::ez(I), ri = R::index(I);
        if constexpr (ez > 0) return up_of(z)[ri * NT + own];
        else if constexpr (ez == 0) return mid_of(z)[ri * NT + own];
        else return dn[ri * NT + own];
    }
};

template <typename T, int Q, bool WALLS, int HVAR, int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 2) hydro_mom_push_kernel(const MomHydroArgs<T> a, int zchunk)
{
    using TL = MomTile<TX, TY, 4>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sphi = reinterpret_cast<T*>(smem_raw);      // [4][TILE] phi ring, then the role arrays
    const Geom& g = a.h.g;
    const size_t N = a.h.N;
    MarchSetup<TL> ms;
    ms.init(g, zchunk);
    if (ms.zb >= ms.ze) return;
    PushBuffers<T, Q, TX, TY> pb;
    pb.init(sphi + 4 * TL::TILE, ms.zb, ms.ze);
    PushSources<TX, TY> ps;
    ps.init(g);
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int own = ty * TX + tx, ownphi = (ty + 1) * TL::PITCH + tx + 2;
    const unsigned inside = PushBuffers<T, Q, TX, TY>::inside_mask(tx, ty);
    const T* const phibase[1] = {a.h.C};
    // "everyone has read the arrays of plane z" is a split barrier: a thread arrives as soon as its Q populations are in
    // registers and waits only before it overwrites arrays in the next expansion, so the arithmetic of the slower warps
    // overlaps the next expansion of the faster ones
    __shared__ unsigned long long pulled;
    if (tx == 0 && ty == 0) mbar_init(&pulled, TX * TY);
    __syncthreads();

    T kq[10], hq[10];      // coefficients of the thread's source entries of the plane to be expanded next
    auto request = [&](int zz) {
        const size_t off = ms.zoff(g, zz);
#pragma unroll
        for (int f = 0; f < 10; ++f) kq[f] = ld_here(a.Ksrc + (size_t)f * N + off + ps.own_src);
        if (ps.kind) {
#pragma unroll
            for (int f = 0; f < 10; ++f) hq[f] = ld_here(a.Ksrc + (size_t)f * N + off + ps.halo_src);
        }
    };
    auto expand = [&](int p) {
        pb.push(p, own, inside, kq[0], kq[1], kq[2], kq[3], kq[4], kq[5], kq[6], kq[7], kq[8], kq[9]);
        if (ps.kind == 1) pb.template push_from_halo<0, 1>(p, ps.hx, ps.hy, hq);
        else if (ps.kind == 2) pb.template push_from_halo<0, -1>(p, ps.hx, ps.hy, hq);
        else if (ps.kind == 3) pb.template push_from_halo<1, 0>(p, ps.hx, ps.hy, hq);
        else if (ps.kind == 4) pb.template push_from_halo<-1, 0>(p, ps.hx, ps.hy, hq);
        else if (ps.kind == 5) {
            if (ps.hx < 0 && ps.hy < 0) pb.template push_from_halo<1, 1>(p, ps.hx, ps.hy, hq);
            else if (ps.hx < 0) pb.template push_from_halo<1, -1>(p, ps.hx, ps.hy, hq);
            else if (ps.hy < 0) pb.template push_from_halo<-1, 1>(p, ps.hx, ps.hy, hq);
            else pb.template push_from_halo<-1, -1>(p, ps.hx, ps.hy, hq);
        }
    };
    for (int zz = ms.zb - 1; zz <= ms.zb + 1; ++zz) ms.load_plane(sphi + ms.slot_of(zz) * TL::TILE, phibase, g, zz);
    cp_async_commit();
    request(ms.zb - 1); expand(ms.zb - 1);
    request(ms.zb); expand(ms.zb);
    request(ms.zb + 1);

    WallFlags wf;
    wf.wxm = WALLS && (g.walls & ACM_WALL_X) && ms.x == 0; wf.wxp = WALLS && (g.walls & ACM_WALL_X) && ms.x == g.nx - 1;
    wf.wym = WALLS && (g.walls & ACM_WALL_Y) && ms.y == 0; wf.wyp = WALLS && (g.walls & ACM_WALL_Y) && ms.y == g.ny - 1;
    const unsigned col = ms.active ? (unsigned)(ms.y * g.nx + ms.x) : 0u;
    for (int z = ms.zb; z < ms.ze; ++z) {
        if (z > ms.zb) mbar_wait(&pulled, (unsigned)(z - 1 - ms.zb) & 1u);      // everyone has read plane z-1: its arrays take this expansion
        expand(z + 1);
        const unsigned idx = (unsigned)z * ms.plane + col;
        const T uox = ld_here(a.Uin + idx), uoy = ld_here(a.Uin + N + idx), uoz = ld_here(a.Uin + 2 * N + idx);
        cp_async_wait_all();
        __syncthreads();      // plane z is complete, the phi planes z-1 .. z+1 have landed
        if (z + 2 <= ms.ze) ms.load_plane(sphi + ms.slot_of(z + 2) * TL::TILE, phibase, g, z + 2);
        cp_async_commit();
        if (!ms.active) mbar_arrive(&pulled);
        if (ms.active) {
            T gp[Q];
            static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; gp[i] = pb.template pull<i>(z, own); });
            mbar_arrive(&pulled);
            if constexpr (WALLS) {
                wf.wzm = (g.walls & WALL_ZLO) && z == g.zlo; wf.wzp = (g.walls & WALL_ZHI) && z == g.zhi - 1;
                if (wf.wxm | wf.wxp | wf.wym | wf.wyp | wf.wzm | wf.wzp) {
                    const OwnK<T> self{a.Ksrc, N, idx};
                    static_for<1, Q>([&](auto ic) {
                        constexpr int i = decltype(ic)::value;
                        constexpr int ex = Lat<Q>::ex(i), ey = Lat<Q>::ey(i), ez = Lat<Q>::ez(i);
                        if (wf.template beyond<-ex, -ey, -ez, true>()) gp[i] = T(Lat<Q>::w(i)) * mom_pull_g<Q, i, T, true, false>(self, wf);
                    });
                }
            }
            TilePhi<T, TL> ph;
            ph.s = sphi;
#pragma unroll
            for (int d = 0; d < 3; ++d) ph.base[d] = ms.slot_of(z - 1 + d) * TL::TILE + ownphi;
            const T c0 = ph.template get<0, 0, 0>();
            T gpx, gpy, gpz, lap;
            fd_phi_acc<Q, T, true>(ph, c0, gpx, gpy, gpz, lap);
            Moments<Q, T, true> m;
            m.compute(gp);
            if (z + 2 <= ms.ze) request(z + 2);      // the populations are consumed: their registers take the next plane's coefficients
            const HydroCell<T> hc = hydro_velocity<T, Q, HVAR>(m, c0, gpx, gpy, gpz, lap, uox, uoy, uoz, a.h);
            a.Uout[idx] = hc.ux; a.Uout[N + idx] = hc.uy; a.Uout[2 * N + idx] = hc.uz;
            const Coeffs<T> k = hydro_coeffs<T, Q, HVAR>(m, hc, a.h);
            T* o = a.Kdst + idx;
            o[0] = k.A; o[N] = k.bx; o[2 * N] = k.by; o[3 * N] = k.bz;
            o[4 * N] = k.Txx; o[5 * N] = k.Tyy; o[6 * N] = k.Tzz; o[7 * N] = k.Txy; o[8 * N] = k.Txz; o[9 * N] = k.Tyz;
        } else if (z + 2 <= ms.ze) request(z + 2);
    }
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
    const GlobalM<T> acc{M, C, Uo, N, &nb};
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        out[(size_t)i * N + idx] = T(Lat<Q>::w(i)) * mom_pull_h<Q, i, T, false, true>(acc, nb);
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
    const GlobalK<T> acc{K, N, &nb};
    T f[Q];
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        f[i] = T(Lat<Q>::w(i)) * mom_pull_g<Q, i, T, true, LOCAL>(acc, nb);
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

// marching kernels: 32 x 8 tiles of columns, `zchunk` planes per block
constexpr int MARCH_TX = 32, MARCH_TY = 8;

template <typename K>
static cudaError_t march_smem(K kernel, size_t bytes)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

static Launch march_launch(const Geom& g, int zchunk, cudaStream_t stream)
{
    const int planes = g.lz1 - g.lz0;
    return Launch{dim3((g.nx + MARCH_TX - 1) / MARCH_TX, (g.ny + MARCH_TY - 1) / MARCH_TY, (planes + zchunk - 1) / zchunk), dim3(MARCH_TX, MARCH_TY, 1), stream};
}

template <typename T>
cudaError_t launch_phase_mom_march(int Q, bool walls, int zchunk, cudaStream_t stream, const MomPhaseArgs<T>& a)
{
    using TL = MomTile<MARCH_TX, MARCH_TY>;
    const size_t bytes = (size_t)TL::RING * 8 * TL::TILE * sizeof(T);
    const Launch l = march_launch(a.g, zchunk, stream);
    cudaError_t e = cudaSuccess;
    ACM_MOM_DISPATCH_Q(Q, QQ, {
        if (walls) { auto k = phase_mom_march_kernel<T, QQ, true, MARCH_TX, MARCH_TY>; e = march_smem(k, bytes); if (e == cudaSuccess) k<<<l.grid, l.block, bytes, l.stream>>>(a, zchunk); }
        else { auto k = phase_mom_march_kernel<T, QQ, false, MARCH_TX, MARCH_TY>; e = march_smem(k, bytes); if (e == cudaSuccess) k<<<l.grid, l.block, bytes, l.stream>>>(a, zchunk); }
    });
    return e != cudaSuccess ? e : cudaGetLastError();
}

template <typename T, int Q, bool WALLS, int HVAR>
static cudaError_t launch_hydro_mom_march_v(int zchunk, cudaStream_t stream, const MomHydroArgs<T>& a)
{
    using TL = MomTile<MARCH_TX, MARCH_TY, 3>;
    const size_t bytes = (size_t)3 * 11 * TL::TILE * sizeof(T);
    const Launch l = march_launch(a.h.g, zchunk, stream);
    auto k = hydro_mom_march_kernel<T, Q, WALLS, HVAR, MARCH_TX, MARCH_TY>;
    cudaError_t e = march_smem(k, bytes);
    if (e == cudaSuccess) k<<<l.grid, l.block, bytes, l.stream>>>(a, zchunk);
    return e != cudaSuccess ? e : cudaGetLastError();
}

template <typename T, int Q, bool WALLS, int HVAR>
static cudaError_t launch_hydro_mom_push_v(int zchunk, cudaStream_t stream, const MomHydroArgs<T>& a)
{
    using TL = MomTile<MARCH_TX, MARCH_TY, 4>;
    const size_t bytes = (size_t)(4 * TL::TILE + PushBuffers<T, Q, MARCH_TX, MARCH_TY>::DOUBLES) * sizeof(T);
    const Launch l = march_launch(a.h.g, zchunk, stream);
    auto k = hydro_mom_push_kernel<T, Q, WALLS, HVAR, MARCH_TX, MARCH_TY>;
    cudaError_t e = march_smem(k, bytes);
    if (e == cudaSuccess) k<<<l.grid, l.block, bytes, l.stream>>>(a, zchunk);
    return e != cudaSuccess ? e : cudaGetLastError();
}

// D3Q15 / D3Q19: the pushing kernel; D3Q27: its role arrays (108 KB) leave room for one block per SM only and the
// marching kernel is 3x faster there (measured, profiles/r2b_profiles.md section 3); D2Q9 comes here only when acm_set_moment_kernels forces it (acm.cu: direct kernels by default)
template <typename T, int Q, bool WALLS>
static cudaError_t launch_hydro_mom_march_q(int zchunk, cudaStream_t stream, const MomHydroArgs<T>& a)
{
    const bool var = a.h.bulk_one || a.h.subiter > 1;
    if constexpr (Q == 15 || Q == 19) {
        if (var) return launch_hydro_mom_push_v<T, Q, WALLS, 1>(zchunk, stream, a);
        return launch_hydro_mom_push_v<T, Q, WALLS, 0>(zchunk, stream, a);
    } else {
        if (var) return launch_hydro_mom_march_v<T, Q, WALLS, 1>(zchunk, stream, a);
        return launch_hydro_mom_march_v<T, Q, WALLS, 0>(zchunk, stream, a);
    }
}

template <typename T>
cudaError_t launch_hydro_mom_march(int Q, bool walls, int zchunk, cudaStream_t stream, const MomHydroArgs<T>& a)
{
    cudaError_t e = cudaSuccess;
    ACM_MOM_DISPATCH_Q(Q, QQ, {
        if (walls) e = launch_hydro_mom_march_q<T, QQ, true>(zchunk, stream, a);
        else e = launch_hydro_mom_march_q<T, QQ, false>(zchunk, stream, a);
    });
    return e;
}

template cudaError_t launch_phase_mom_march<ACM_T>(int, bool, int, cudaStream_t, const MomPhaseArgs<ACM_T>&);
template cudaError_t launch_hydro_mom_march<ACM_T>(int, bool, int, cudaStream_t, const MomHydroArgs<ACM_T>&);
template cudaError_t launch_phase_mom<ACM_T>(int, bool, const Launch&, const MomPhaseArgs<ACM_T>&);
template cudaError_t launch_hydro_mom<ACM_T>(int, bool, bool, const Launch&, const MomHydroArgs<ACM_T>&);
template cudaError_t launch_init_mom<ACM_T>(const Launch&, const ACM_T*, const ACM_T*, ACM_T*, ACM_T*, ACM_T*, ACM_T*, ACM_T*, Geom, size_t);
template cudaError_t launch_export_h_mom<ACM_T>(int, const Launch&, const ACM_T*, const ACM_T*, const ACM_T*, ACM_T*, Geom, size_t);
template cudaError_t launch_export_g_mom<ACM_T>(int, bool, const Launch&, const ACM_T*, const ACM_T*, ACM_T*, ACM_T*, Geom, size_t, ACM_T, ACM_T);

}  // namespace acm
