// lattice.cuh -- compile-time D2Q9/D3Q15/D3Q19/D3Q27 tables and the two shared "moment <-> population"
// building blocks of the ACM kernels (no runtime tables: everything folds into immediates).
//
// Canonical direction order (include/acm.h): rest; axis pairs; edge pairs; corner pairs; the
// opposite of an odd index k is k+1.  Weights are the textbook ones of the lattices the paper
// names.
#pragma once
#include <type_traits>

namespace acm {

__host__ __device__ constexpr int dir27(int k, int a)
{
    constexpr signed char t[27][3] = {
        {0, 0, 0},
        {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1},
        {1, 1, 0}, {-1, -1, 0}, {1, -1, 0}, {-1, 1, 0},
        {1, 0, 1}, {-1, 0, -1}, {1, 0, -1}, {-1, 0, 1},
        {0, 1, 1}, {0, -1, -1}, {0, 1, -1}, {0, -1, 1},
        {1, 1, 1}, {-1, -1, -1}, {1, 1, -1}, {-1, -1, 1},
        {1, -1, 1}, {-1, 1, -1}, {-1, 1, 1}, {1, -1, -1}};
    return t[k][a];
}

template <int Q>
struct Lat {
    static_assert(Q == 9 || Q == 15 || Q == 19 || Q == 27, "unsupported lattice");
    // D2Q9: the nine directions of the x-y plane, on a grid with one z plane
    static constexpr int DIM = Q == 9 ? 2 : 3;
    // index into the 27-direction list
    __host__ __device__ static constexpr int k27(int i) { return (Q == 15 && i >= 7) ? i + 12 : (Q == 9 && i >= 5) ? i + 2 : i; }
    __host__ __device__ static constexpr int ex(int i) { return dir27(k27(i), 0); }
    __host__ __device__ static constexpr int ey(int i) { return dir27(k27(i), 1); }
    __host__ __device__ static constexpr int ez(int i) { return dir27(k27(i), 2); }
    // |e|^2: 0 rest, 1 axis, 2 edge, 3 corner
    __host__ __device__ static constexpr int cls(int i) { return ex(i) * ex(i) + ey(i) * ey(i) + ez(i) * ez(i); }
    __host__ __device__ static constexpr int opp(int i) { return i == 0 ? 0 : ((i & 1) ? i + 1 : i - 1); }
    // weight of a class
    __host__ __device__ static constexpr double wc(int c)
    {
        return Q == 9  ? (c == 0 ? 4.0 / 9.0 : c == 1 ? 1.0 / 9.0 : 1.0 / 36.0)
             : Q == 15 ? (c == 0 ? 2.0 / 9.0 : c == 1 ? 1.0 / 9.0 : 1.0 / 72.0)
             : Q == 19 ? (c == 0 ? 1.0 / 3.0 : c == 1 ? 1.0 / 18.0 : 1.0 / 36.0)
                       : (c == 0 ? 8.0 / 27.0 : c == 1 ? 2.0 / 27.0 : c == 2 ? 1.0 / 54.0 : 1.0 / 216.0);
    }
    __host__ __device__ static constexpr double w(int i) { return wc(cls(i)); }
    __host__ __device__ static constexpr bool has_cls(int c) { return c <= 1 || (c == 2 && Q != 15) || (c == 3 && Q != 19 && Q != 9); }
};

template <int I, int N, int S = 1, typename F>
__device__ __forceinline__ void static_for(F&& f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + S, N, S>(f);
    }
}

// acc += s * v with s in {-1,0,1} known at compile time
template <int S, typename T>
__device__ __forceinline__ void addsgn(T& acc, T v)
{
    if constexpr (S > 0) acc += v;
    else if constexpr (S < 0) acc -= v;
}

// Moments of a population set f[Q] up to second order:
//   m0 = sum f, j = sum f e, P_ab = sum f e_a e_b       (pair sums/differences shared)
template <int Q, typename T, bool SECOND>
struct Moments {
    T m0, jx, jy, jz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz;
    __device__ __forceinline__ void compute(const T (&f)[Q])
    {
        using L = Lat<Q>;
        m0 = f[0];
        jx = jy = jz = T(0);
        Pxx = Pyy = Pzz = Pxy = Pxz = Pyz = T(0);
        static_for<1, Q, 2>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            constexpr int ex = L::ex(i), ey = L::ey(i), ez = L::ez(i);
            const T s = f[i] + f[i + 1];
            const T d = f[i] - f[i + 1];
            m0 += s;
            addsgn<ex>(jx, d); addsgn<ey>(jy, d); addsgn<ez>(jz, d);
            if constexpr (SECOND) {
                addsgn<ex * ex>(Pxx, s); addsgn<ey * ey>(Pyy, s); addsgn<ez * ez>(Pzz, s);
                addsgn<ex * ey>(Pxy, s); addsgn<ex * ez>(Pxz, s); addsgn<ey * ez>(Pyz, s);
            }
        });
    }
};

// Populations of the form  f_i = w_i [ A + e_i.b + e_ia e_ib T_ab ]  (T symmetric), which is what
// both closed-form collisions reduce to.  Per class the scalars are pre-scaled by the weight;
// per opposite pair the even part E and the odd part O are shared: f_i = E + O, f_ibar = E - O.
template <int Q, typename T, typename Store>
__device__ __forceinline__ void emit_populations(T A, T bx, T by, T bz, T Txx, T Tyy, T Tzz, T Txy, T Txz, T Tyz,
                                                 Store&& store)
{
    using L = Lat<Q>;
    store(std::integral_constant<int, 0>{}, T(L::wc(0)) * A);
    static_for<1, 4>([&](auto cc) {
        constexpr int c = decltype(cc)::value;
        if constexpr (L::has_cls(c)) {
            constexpr T w = T(L::wc(c));
            const T Ac = w * A, bxc = w * bx, byc = w * by, bzc = w * bz;
            const T Txxc = w * Txx, Tyyc = w * Tyy, Tzzc = w * Tzz;
            const T Txyc = T(2) * w * Txy, Txzc = T(2) * w * Txz, Tyzc = T(2) * w * Tyz;
            static_for<1, Q, 2>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                if constexpr (L::cls(i) == c) {
                    constexpr int ex = L::ex(i), ey = L::ey(i), ez = L::ez(i);
                    T E = Ac;                      // same expression tree for pairs with the same support => CSE
                    addsgn<ex * ex>(E, Txxc); addsgn<ey * ey>(E, Tyyc); addsgn<ez * ez>(E, Tzzc);
                    addsgn<ex * ey>(E, Txyc); addsgn<ex * ez>(E, Txzc); addsgn<ey * ez>(E, Tyzc);
                    T O = T(0);
                    bool first = true;
                    auto odd = [&](auto sc, T v) {
                        constexpr int s = decltype(sc)::value;
                        if constexpr (s != 0) {
                            if (first) { O = (s > 0) ? v : -v; first = false; }
                            else addsgn<s>(O, v);
                        }
                    };
                    odd(std::integral_constant<int, ex>{}, bxc);
                    odd(std::integral_constant<int, ey>{}, byc);
                    odd(std::integral_constant<int, ez>{}, bzc);
                    store(std::integral_constant<int, i>{}, E + O);
                    store(std::integral_constant<int, i + 1>{}, E - O);
                }
            });
        }
    });
}

}  // namespace acm
