// pair.cuh -- geometry, streaming and phi-stencil access for the kernels that update TWO x-adjacent cells
// (x0, x0 + 1), x0 even, per thread (element type vec2<S>, vec2.cuh).  The own-cell accesses and every pull /
// push along a direction with e_x = 0 are ONE aligned 8-byte (fp32) or 16-byte (fp64) access; a direction with
// e_x = +-1 shifts the pair by one element, which breaks the alignment: two scalar accesses.  Needs nx even (rows
// and population planes then start on an even element).  Mirrors Nbr / load_incoming / outgoing_ptr / PhiGlobal
// of common.cuh, which stay the single-cell path.
#pragma once
#include "common.cuh"
#include "vec2.cuh"

namespace acm {

template <typename S> struct native2;
template <> struct native2<float> { using type = float2; };
template <> struct native2<double> { using type = double2; };

template <typename S> __device__ __forceinline__ vec2<S> ld_pair(const S* p)      // p: even element
{
    return vec2<S>(*reinterpret_cast<const typename native2<S>::type*>(p));
}
template <typename S> __device__ __forceinline__ vec2<S> ldg_pair(const S* p)
{
    return vec2<S>(__ldg(reinterpret_cast<const typename native2<S>::type*>(p)));
}
template <typename S> __device__ __forceinline__ void st_pair(S* p, vec2<S> v)
{
    *reinterpret_cast<typename native2<S>::type*>(p) = v.v;
}

// pair of the calling thread: 3-D launch (block tiles of x-rows, blockDim.x threads = 2 blockDim.x cells) or linear
// launch over the pairs of the planes [lz0, lz1)
__device__ __forceinline__ bool pair_of_thread(const Geom& g, int& x0, int& y, int& z)
{
    const unsigned hx = (unsigned)g.nx >> 1;
    if (g.linear) {
        const unsigned id = blockIdx.x * blockDim.x + threadIdx.x;
        if (id >= hx * (unsigned)g.ny * (unsigned)(g.lz1 - g.lz0)) return false;
        const unsigned t = id / hx;
        x0 = (int)(2u * (id - t * hx));
        const unsigned zr = t / (unsigned)g.ny;
        y = (int)(t - zr * (unsigned)g.ny);
        z = g.lz0 + (int)zr;
        return true;
    }
    x0 = 2 * (int)(blockIdx.x * blockDim.x + threadIdx.x);
    y = blockIdx.y * blockDim.y + threadIdx.y;
    z = g.lz0 + blockIdx.z * blockDim.z + threadIdx.z;
    return x0 < g.nx && y < g.ny && z < g.lz1;
}

// Neighbourhood of the pair (x0, x0+1): the element left of it (x0 - 1) and right of it (x0 + 2) with periodic wrap
// or, at a wall, clamped (= the mirror ghost of the phi stencil); rows and "beyond a wall" flags as in Nbr.  Only
// the first cell can have its x - 1 neighbour beyond a wall, only the second its x + 1 neighbour.
struct Nbr2 {
    unsigned xm, x0, xp;
    unsigned row[3][3];
    bool wxm, wxp, wym, wyp, wzm, wzp;
    bool peer_lo, peer_hi;

    template <bool WALLS>
    __device__ __forceinline__ void setup(const Geom& g, int x, int y, int z)
    {
        wxm = wxp = wym = wyp = wzm = wzp = false;
        int l = x - 1, r = x + 2, ym = y - 1, yp = y + 1, zm = z - 1, zp = z + 1;
        if (l < 0) { if (WALLS && (g.walls & ACM_WALL_X)) { wxm = true; l = 0; } else l = g.nx - 1; }
        if (r >= g.nx) { if (WALLS && (g.walls & ACM_WALL_X)) { wxp = true; r = g.nx - 1; } else r = 0; }
        if (ym < 0) { if (WALLS && (g.walls & ACM_WALL_Y)) { wym = true; ym = 0; } else ym = g.ny - 1; }
        if (yp >= g.ny) { if (WALLS && (g.walls & ACM_WALL_Y)) { wyp = true; yp = g.ny - 1; } else yp = 0; }
        if (zm < g.zlo) { if (WALLS && (g.walls & WALL_ZLO)) { wzm = true; zm = g.zlo; } else if (!g.zghost) zm = g.zhi - 1; }
        if (zp >= g.zhi) { if (WALLS && (g.walls & WALL_ZHI)) { wzp = true; zp = g.zhi - 1; } else if (!g.zghost) zp = g.zlo; }
        peer_lo = g.zghost && z == g.zlo && !wzm;
        peer_hi = g.zghost && z == g.zhi - 1 && !wzp;
        xm = (unsigned)l; x0 = (unsigned)x; xp = (unsigned)r;
        const int ys[3] = {ym, y, yp}, zs[3] = {zm, z, zp};
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) row[a][b] = (unsigned)((zs[a] * g.ny + ys[b]) * g.nx);
    }
    // element index of cell K (0: x0, 1: x0 + 1) of the pair, shifted by (dx, dy, dz)
    template <int K, int DX, int DY, int DZ>
    __device__ __forceinline__ unsigned at() const
    {
        const unsigned r = row[DZ + 1][DY + 1];
        if constexpr (DX == 0) return r + x0 + K;
        else if constexpr (DX < 0) return r + (K == 0 ? xm : x0);
        else return r + (K == 0 ? x0 + 1 : xp);
    }
    __device__ __forceinline__ unsigned own() const { return row[1][1] + x0; }      // even: aligned pair
    template <int K, int DX, int DY, int DZ, bool WALLS>
    __device__ __forceinline__ bool beyond() const
    {
        if constexpr (!WALLS) return false;
        bool b = false;
        if constexpr (DX < 0 && K == 0) b |= wxm;
        if constexpr (DX > 0 && K == 1) b |= wxp;
        if constexpr (DY < 0) b |= wym;
        if constexpr (DY > 0) b |= wyp;
        if constexpr (DZ < 0) b |= wzm;
        if constexpr (DZ > 0) b |= wzp;
        return b;
    }
};

// incoming populations f_i of both cells from an array in state STATE (see load_incoming)
template <int Q, typename S, bool WALLS, int STATE, bool PEER = false>
__device__ __forceinline__ void load_incoming2(const S* F, size_t N, const Nbr2& nb, vec2<S> (&f)[Q], Peers<S> peers = Peers<S>{nullptr, nullptr})
{
    using L = Lat<Q>;
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int ex = L::ex(i), ey = L::ey(i), ez = L::ez(i), o = L::opp(i);
        if constexpr (STATE == ST_IN) {
            f[i] = ld_pair(F + (size_t)i * N + nb.own());
        } else {
            constexpr int far = (STATE == ST_POST) ? i : o;      // slot at x - e_i
            constexpr int own = (STATE == ST_POST) ? o : i;      // slot at x when x - e_i is beyond a wall
            const S* base = F;
            if constexpr (PEER && ez > 0) base = nb.peer_lo ? peers.lo : F;      // pulled from the plane z - 1
            if constexpr (PEER && ez < 0) base = nb.peer_hi ? peers.hi : F;      // pulled from the plane z + 1
            if constexpr (ex == 0) {
                const S* src = base + (size_t)far * N + nb.template at<0, 0, -ey, -ez>();
                if constexpr (WALLS && i > 0) {
                    if (nb.template beyond<0, 0, -ey, -ez, WALLS>()) src = F + (size_t)own * N + nb.own();
                }
                f[i] = ld_pair(src);
            } else {
                const S* s0 = base + (size_t)far * N + nb.template at<0, -ex, -ey, -ez>();
                const S* s1 = base + (size_t)far * N + nb.template at<1, -ex, -ey, -ez>();
                if constexpr (WALLS) {
                    if (nb.template beyond<0, -ex, -ey, -ez, WALLS>()) s0 = F + (size_t)own * N + nb.own();
                    if (nb.template beyond<1, -ex, -ey, -ez, WALLS>()) s1 = F + (size_t)own * N + nb.own() + 1;
                }
                f[i] = vec2<S>(*s0, *s1);
            }
        }
    });
}

// store of the post-collision populations f*_I of both cells into the array the step writes (see outgoing_ptr)
template <int Q, int I, typename S, bool WALLS, int FROM>
__device__ __forceinline__ void store_outgoing2(S* F, size_t N, const Nbr2& nb, vec2<S> v)
{
    using L = Lat<Q>;
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I), o = L::opp(I);
    if constexpr (FROM == ST_POST) {
        st_pair(F + (size_t)I * N + nb.own(), v);
    } else if constexpr (FROM == ST_IN) {
        st_pair(F + (size_t)o * N + nb.own(), v);
    } else if constexpr (ex == 0) {
        S* dst = F + (size_t)I * N + nb.template at<0, 0, ey, ez>();
        if constexpr (WALLS && I > 0) {
            if (nb.template beyond<0, 0, ey, ez, WALLS>()) dst = F + (size_t)o * N + nb.own();
        }
        st_pair(dst, v);
    } else {
        S* d0 = F + (size_t)I * N + nb.template at<0, ex, ey, ez>();
        S* d1 = F + (size_t)I * N + nb.template at<1, ex, ey, ez>();
        if constexpr (WALLS) {
            if (nb.template beyond<0, ex, ey, ez, WALLS>()) d0 = F + (size_t)o * N + nb.own();
            if (nb.template beyond<1, ex, ey, ez, WALLS>()) d1 = F + (size_t)o * N + nb.own() + 1;
        }
        *d0 = v.v.x;
        *d1 = v.v.y;
    }
}

// phi stencil of the pair through L1/L2.  The four values of a row (x0 - 1 .. x0 + 2) serve the three x-shifts of
// both cells: one aligned pair load (the compiler merges its repeats) and one scalar load per side.
template <typename S, bool PEER = false>
struct PhiGlobal2 {
    const S* C;
    const Nbr2* nb;
    Peers<S> peers;
    template <int DX, int DY, int DZ> __device__ __forceinline__ vec2<S> get() const
    {
        const S* base = C;
        if constexpr (PEER && DZ < 0) base = nb->peer_lo ? peers.lo : C;
        if constexpr (PEER && DZ > 0) base = nb->peer_hi ? peers.hi : C;
        const vec2<S> mid = ldg_pair(base + nb->template at<0, 0, DY, DZ>());
        if constexpr (DX == 0) return mid;
        else if constexpr (DX < 0) return vec2<S>(__ldg(base + nb->template at<0, -1, DY, DZ>()), mid.v.x);
        else return vec2<S>(mid.v.y, __ldg(base + nb->template at<1, 1, DY, DZ>()));
    }
};

}  // namespace acm
