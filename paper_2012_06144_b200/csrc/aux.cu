// aux.cu -- the light kernels of libacm: equilibrium initialiser, export / import of the
// populations in the ABI's conventions, deterministic block reductions (sum of phi, bubble
// diagnostics).  Both precisions are instantiated here.
#include "kernels.h"

namespace acm {

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

// Gamma_i(u) - w_i without the cancellation
template <int Q, typename T>
__device__ __forceinline__ T gamma_dev(int ex, int ey, int ez, T w, T ux, T uy, T uz)
{
    const T eu = T(ex) * ux + T(ey) * uy + T(ez) * uz;
    return w * (T(3) * eu + T(4.5) * eu * eu - T(1.5) * (ux * ux + uy * uy + uz * uz));
}

// ref: reference phase of the fp32 deviation storage (C <- phi - ref, h <- h - ref w_i; A22); 0 for fp64
template <typename T, int QH, int QG, bool INPLACE>
__global__ void init_kernel(const T* __restrict__ phi, const T* __restrict__ u, T* H, T* G, T* C, T* U, Geom g, size_t N, T ref)
{
    int x, y, z;
    if (!cell_of_thread(g, x, y, z)) return;
    Nbr nb;
    nb.setup<true>(g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    const T ph = phi[idx];
    const T ux = u[idx], uy = u[N + idx], uz = u[2 * N + idx];
    C[idx] = ph - ref;
    U[idx] = ux; U[N + idx] = uy; U[2 * N + idx] = uz;
    static_for<0, QH>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        using L = Lat<QH>;
        constexpr int slot = INPLACE ? L::opp(i) : i;
        if constexpr (sizeof(T) == 4)      // phi Gamma - ref w = (phi - ref) Gamma + ref (Gamma - w)
            H[(size_t)slot * N + idx] = (ph - ref) * gamma_i<QH, T>(L::ex(i), L::ey(i), L::ez(i), T(L::w(i)), ux, uy, uz) +
                                        ref * gamma_dev<QH, T>(L::ex(i), L::ey(i), L::ez(i), T(L::w(i)), ux, uy, uz);
        else
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
            const unsigned j = nb.template at<ex, ey, ez>();
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
__global__ void export_kernel(const T* F, const T* __restrict__ C, T* out, T* p, Geom g, size_t N, T rho_L, T drho, T shift)
{
    int x, y, z;
    if (!cell_of_thread(g, x, y, z)) return;
    Nbr nb;
    nb.setup<true>(g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    T f[Q];
    if constexpr (POST) static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; f[i] = load_post<Q, i, T, STATE>(F, N, nb); });
    else load_incoming<Q, T, true, STATE>(F, N, nb, f);
    // shift: the array holds f_i - shift w_i (fp32 deviation storage of h); rho_L is rho at the reference phase
    if (out) static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        out[(size_t)i * N + idx] = shift != T(0) ? f[i] + shift * T(Lat<Q>::w(i)) : f[i];
    });
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
__global__ void import_kernel(const T* __restrict__ in, T* F, Geom g, size_t N, T shift)
{
    int x, y, z;
    if (!cell_of_thread(g, x, y, z)) return;
    Nbr nb;
    nb.setup<true>(g, x, y, z);
    const unsigned idx = nb.at<0, 0, 0>();
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        using L = Lat<Q>;
        constexpr int ex = L::ex(i), ey = L::ey(i), ez = L::ez(i);
        if constexpr (POST) {
            const T v = in[(size_t)i * N + idx];
            F[(size_t)L::opp(i) * N + idx] = shift != T(0) ? v - shift * T(L::w(i)) : v;
        } else {
            const T v = nb.template beyond<ex, ey, ez, true>() ? in[(size_t)L::opp(i) * N + idx]
                                                               : in[(size_t)i * N + nb.template at<ex, ey, ez>()];
            F[(size_t)i * N + idx] = v;
        }
    });
}

// out_i = in_i + shift w_i on the owned cells (conversion between the ABI's h and the fp32 deviation storage)
template <typename T, int Q>
__global__ void shift_pop_kernel(const T* __restrict__ in, T* out, Geom g, size_t N, T shift)
{
    int x, y, z;
    if (!cell_of_thread(g, x, y, z)) return;
    const size_t idx = ((size_t)z * g.ny + y) * g.nx + x;
    static_for<0, Q>([&](auto ic) { constexpr int i = decltype(ic)::value; out[(size_t)i * N + idx] = in[(size_t)i * N + idx] + shift * T(Lat<Q>::w(i)); });
}

// out = in + shift (phi from / to its deviation storage), whole array
template <typename T>
__global__ void shift_field_kernel(const T* __restrict__ in, T* out, size_t n, T shift)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) out[i] = in[i] + shift;
}

// deterministic two-pass sum: fixed grid, fixed per-thread order, shuffle tree, fixed final order

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

// Rising-bubble diagnostics (section 6.1; reading A24): seven sums weighted with the
// light-phase weight (1 - phi) [phi < 1/2]:  V, V x_c, V y_c, V z_c (cell centres i + 1/2), V u_x, V u_y, V u_z.
// Same fixed-order two-pass scheme as sum(phi), so the result is bitwise reproducible.
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) diag_pass1(const T* __restrict__ C, const T* __restrict__ U, Geom g, size_t N, int zshift, double ref, double* part)
{
    // cells of the owned planes [zlo, zhi); z coordinate reported in the global frame (slab: + zshift)
    double s[DIAG_WIDTH] = {0, 0, 0, 0, 0, 0, 0};
    const size_t plane = (size_t)g.nx * g.ny;
    const size_t end = (size_t)g.zhi * plane;
    for (size_t i = (size_t)g.zlo * plane + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < end; i += (size_t)gridDim.x * blockDim.x) {
        const int zl = (int)(i / plane);
        const int r = (int)(i - (size_t)zl * plane);
        const int z = zl + zshift;
        const int y = r / g.nx, x = r - y * g.nx;
        const double om = (1.0 - ref) - (double)C[i];     // 1 - phi (C holds phi - ref)
        const double w = om > 0.5 ? om : 0.0;             // cells of the bubble: phi < 1/2
        s[0] += w;
        s[1] += w * (x + 0.5); s[2] += w * (y + 0.5); s[3] += w * (z + 0.5);
        s[4] += w * (double)U[i]; s[5] += w * (double)U[N + i]; s[6] += w * (double)U[2 * N + i];
    }
#pragma unroll
    for (int k = 0; k < DIAG_WIDTH; ++k) {
        const double v = block_sum(s[k]);
        if (threadIdx.x == 0) part[(size_t)k * RED_BLOCKS + blockIdx.x] = v;
        __syncthreads();      // block_sum's shared scratch is reused by the next component
    }
}

// one block per component: fixed-order sum of its RED_BLOCKS partials
__global__ void __launch_bounds__(RED_THREADS) diag_pass2(const double* __restrict__ part, double* out)
{
    double s = 0.0;
    for (int i = threadIdx.x; i < RED_BLOCKS; i += blockDim.x) s += part[(size_t)blockIdx.x * RED_BLOCKS + i];
    s = block_sum(s);
    if (threadIdx.x == 0) out[blockIdx.x] = s;
}

// ------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------
#define ACM_DISPATCH_Q(q, QQ, ...)                                 \
    switch (q) {                                                    \
        case 9: { constexpr int QQ = 9; __VA_ARGS__; } break;       \
        case 15: { constexpr int QQ = 15; __VA_ARGS__; } break;     \
        case 19: { constexpr int QQ = 19; __VA_ARGS__; } break;     \
        default: { constexpr int QQ = 27; __VA_ARGS__; } break;     \
    }

#define ACM_DISPATCH_Q3(q, QQ, ...)                                \
    switch (q) {                                                    \
        case 15: { constexpr int QQ = 15; __VA_ARGS__; } break;     \
        case 19: { constexpr int QQ = 19; __VA_ARGS__; } break;     \
        default: { constexpr int QQ = 27; __VA_ARGS__; } break;     \
    }

template <typename T>
cudaError_t launch_init(int Qh, int Qg, bool inplace, const Launch& l, const T* phi, const T* u, T* H, T* G, T* C, T* U, Geom g, size_t N, T ref)
{
    if (Qh == 9 || Qg == 9) {       // the two-dimensional instance uses D2Q9 for both steps
        if (inplace) init_kernel<T, 9, 9, true><<<l.grid, l.block, 0, l.stream>>>(phi, u, H, G, C, U, g, N, ref);
        else init_kernel<T, 9, 9, false><<<l.grid, l.block, 0, l.stream>>>(phi, u, H, G, C, U, g, N, ref);
        return cudaGetLastError();
    }
    ACM_DISPATCH_Q3(Qh, QH, ACM_DISPATCH_Q3(Qg, QG, {
        if (inplace) init_kernel<T, QH, QG, true><<<l.grid, l.block, 0, l.stream>>>(phi, u, H, G, C, U, g, N, ref);
        else init_kernel<T, QH, QG, false><<<l.grid, l.block, 0, l.stream>>>(phi, u, H, G, C, U, g, N, ref);
    }));
    return cudaGetLastError();
}

template <typename T, int Q, bool POST>
static void export_state(int state, const Launch& l, const T* F, const T* C, T* out, T* p, Geom g, size_t N, T rho_L, T drho, T shift)
{
    if (state == ST_POST) export_kernel<T, Q, ST_POST, POST><<<l.grid, l.block, 0, l.stream>>>(F, C, out, p, g, N, rho_L, drho, shift);
    else if (state == ST_IN) export_kernel<T, Q, ST_IN, POST><<<l.grid, l.block, 0, l.stream>>>(F, C, out, p, g, N, rho_L, drho, shift);
    else export_kernel<T, Q, ST_SWAP, POST><<<l.grid, l.block, 0, l.stream>>>(F, C, out, p, g, N, rho_L, drho, shift);
}

template <typename T>
cudaError_t launch_export(int Q, int state, bool post, const Launch& l, const T* F, const T* C, T* out, T* p, Geom g, size_t N, T rho_L, T drho, T shift)
{
    ACM_DISPATCH_Q(Q, QQ, {
        if (post) export_state<T, QQ, true>(state, l, F, C, out, p, g, N, rho_L, drho, shift);
        else export_state<T, QQ, false>(state, l, F, C, out, p, g, N, rho_L, drho, shift);
    });
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_import(int Q, bool post, const Launch& l, const T* in, T* F, Geom g, size_t N, T shift)
{
    ACM_DISPATCH_Q(Q, QQ, {
        if (post) import_kernel<T, QQ, true><<<l.grid, l.block, 0, l.stream>>>(in, F, g, N, shift);
        else import_kernel<T, QQ, false><<<l.grid, l.block, 0, l.stream>>>(in, F, g, N, shift);
    });
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_shift_pop(int Q, const Launch& l, const T* in, T* out, Geom g, size_t N, T shift)
{
    ACM_DISPATCH_Q(Q, QQ, { shift_pop_kernel<T, QQ><<<l.grid, l.block, 0, l.stream>>>(in, out, g, N, shift); });
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_shift_field(cudaStream_t s, const T* in, T* out, size_t n, T shift)
{
    shift_field_kernel<T><<<RED_BLOCKS, RED_THREADS, 0, s>>>(in, out, n, shift);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_sum_phi(cudaStream_t s, const T* C, size_t N, double* part)
{
    sum_pass1<T><<<RED_BLOCKS, RED_THREADS, 0, s>>>(C, N, part);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    sum_pass2<<<1, RED_THREADS, 0, s>>>(part, RED_BLOCKS, part + RED_BLOCKS);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_bubble_diag(cudaStream_t s, const T* C, const T* U, Geom g, size_t N, int zshift, double ref, double* part)
{
    diag_pass1<T><<<RED_BLOCKS, RED_THREADS, 0, s>>>(C, U, g, N, zshift, ref, part);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    diag_pass2<<<DIAG_WIDTH, RED_THREADS, 0, s>>>(part, part + (size_t)DIAG_WIDTH * RED_BLOCKS);
    return cudaGetLastError();
}

#define ACM_INSTANTIATE_AUX(T)                                                                                              \
    template cudaError_t launch_init<T>(int, int, bool, const Launch&, const T*, const T*, T*, T*, T*, T*, Geom, size_t, T); \
    template cudaError_t launch_shift_pop<T>(int, const Launch&, const T*, T*, Geom, size_t, T);                             \
    template cudaError_t launch_shift_field<T>(cudaStream_t, const T*, T*, size_t, T);                                      \
    template cudaError_t launch_export<T>(int, int, bool, const Launch&, const T*, const T*, T*, T*, Geom, size_t, T, T, T); \
    template cudaError_t launch_import<T>(int, bool, const Launch&, const T*, T*, Geom, size_t, T);                         \
    template cudaError_t launch_sum_phi<T>(cudaStream_t, const T*, size_t, double*);                                        \
    template cudaError_t launch_bubble_diag<T>(cudaStream_t, const T*, const T*, Geom, size_t, int, double, double*);
ACM_INSTANTIATE_AUX(double)
ACM_INSTANTIATE_AUX(float)

}  // namespace acm
