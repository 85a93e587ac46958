// acm.cu -- libacm host side: context, workspace layout, dispatch to the kernel launchers of
// kernels.h, and the C ABI of include/acm.h.  The kernels are in phase_*.cu, hydro_*.cu, aux.cu.
//
// Storage on the device (all SoA, x fastest, 64-bit offsets for the q planes):
//   H[2][Qh][N]  phase populations, post-collision value at their own cell (pulled by the next step)
//   G[2][Qg][N]  hydrodynamic populations, ALSO stored post-collision at their own cell: the paper's
//                "collide-stream-push" is realised as a pull at the start of the next
//                hydrodynamic step ("lazy pull"); acm_get_pdfs / acm_fields apply the pending
//                streaming, the initialiser pre-shifts g.  Aligned, fully coalesced stores.
//   C[2][N]      phi (double-buffered: the phase kernel reads a stencil of the old phi and writes new)
//   U[3][N]      velocity, in place
// With ACM_OPT_INPLACE there is one H and one G array (AA pattern, see common.cuh).
// With ACM_OPT_MOMENTS the H region holds M[2][4][N] and the G region K[2][10][N] (the coefficients of the
// post-collision state, moment_impl.cuh) and U is double-buffered.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <type_traits>
#include <vector>

#include "kernels.h"

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
    int nx, ny, nz, Qh, Qg, precision;   // nz = allocated planes (owned planes + 2 ghost planes for a slab)
    size_t N, esz;                        // N = nx*ny*nz: the stride between population planes
    // slab of a z-decomposed domain (acm_create_slab); a plain context owns everything: nzl = nz, zlo = 0
    int nzl, zlo, ghost;                  // owned planes [zlo, zlo+nzl), ghost = 1: planes zlo-1 and zlo+nzl are halos
    int zglob0, nz_global, rank, nranks;  // global z of the first owned plane, global height, position in the decomposition
    // peer mode of a slab (acm_set_peers): workspaces of the neighbour slabs, read directly by the LB kernels
    bool peer_on;
    char *peer_lo, *peer_hi;
    // fp32 instance: h and phi are stored as deviations from the reference phase (A22)
    int ref_mode;                         // -1: chosen by acm_init (the majority phase; heavy for slabs), else 0 / 1
    double ref;                           // 0 or 1; always 0 for fp64
    double rho_H, rho_L, sigma, xi, M, nu_H, nu_L, grav[3];
    unsigned walls;
    cudaStream_t stream;
    char* ws;
    // carved workspace (byte offsets)
    size_t offH[2], offG[2], offC[2], offU[2], offStage, offRed;
    int curH, curG, curC, curU;       // which buffer holds the current state
    int uH;                           // ACM_OPT_MOMENTS: the velocity buffer the current coefficients of h* were built with
    int mom_mode, mom_zchunk;         // ACM_OPT_MOMENTS: -1 automatic | 0 direct kernels | 1 marching kernels; planes per block (0 = automatic)
    int sm_count;
    unsigned options;           // ACM_OPT_*
    int stH, stG;               // storage state of the current H / G buffer (ST_POST | ST_IN | ST_SWAP)
    bool initialised;
    int sticky;                 // ACM_OK or ACM_ECUDA
    dim3 block;
    long long launches;
    long long steps_done;       // committed hydrodynamic steps since acm_init (acm_state_signature)
    int cpt_phase, cpt_hydro;   // cells per thread of the two LB kernels: 1, or 2 (pair kernels: 8 / 16-byte accesses, packed fp32)
    int subiter;                // sweeps of the fixed point of eq. 22 (acm_set_subiter; 1 = the single evaluation, A10)
    int phase_planes, hydro_planes;   // owned planes launched since the last acm_*_commit (guard of the split launches)
    // optional per-kernel timing (acm_profile): events recorded around every LB kernel.  The events come from a pool
    // that acm_step fills BEFORE its first launch, so that nothing but cudaEventRecord sits between two kernels.
    bool profiling;
    std::vector<cudaEvent_t> ev;     // pool; the first ev_used are recorded: per acm_step call e0 [phase] e1 [hydro] e2 [phase] ...
    size_t ev_used;
    std::vector<int> ev_calls;       // number of steps of each recorded acm_step call
    // CUDA graphs of GRAPH_STEPS consecutive steps for launch-bound (small) grids (acm_set_graph)
    int graph_mode;                  // -1: automatic (grids of at most GRAPH_AUTO_CELLS cells), 0: never, 1: always
    cudaStream_t cap_stream;         // private stream the steps are captured on (the caller's may be the legacy stream)
    struct GraphEntry { unsigned key; cudaGraphExec_t exec; };
    std::vector<GraphEntry> graphs;  // one per buffer / storage-state parity the capture started from
    long long graph_replays;
    // acm_run_host: the device-to-host copies of the results run on a private stream behind events, so that phi
    // (final after the last phase-field kernel) already travels while the last hydrodynamic kernel runs
    cudaStream_t io_stream;
    cudaEvent_t io_ev[4];
};

// A graph holds an even number of steps: the buffer parity of the two-grid layout and the even/odd kernels of the
// in-place pattern both repeat with period 2, so a replay leaves the host-side state as it found it.
constexpr int GRAPH_STEPS = 16;
constexpr size_t GRAPH_AUTO_CELLS = (size_t)1 << 18;     // 64^3: below this a kernel is as short as its launch

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

static bool valid_stencil(int q) { return q == 9 || q == 15 || q == 19 || q == 27; }

constexpr size_t MOM_H = 4, MOM_G = 10;      // planes of the coefficient arrays M (A, b) and K (A, b, T)

struct Layout {
    size_t offH[2], offG[2], offC[2], offU[2], offStage, offRed, total;
};

static bool make_layout(int nx, int ny, int nz, int Qh, int Qg, int precision, unsigned options, Layout* L)
{
    if (options & ~(unsigned)ACM_OPT_ALL) return false;
    if ((options & ACM_OPT_UNFUSED) && (options & ACM_OPT_INPLACE)) return false;   // Algorithm 1 is a two-grid scheme
    // moment representation: two-grid fused kernels, MRT phase-field collision (SRT keeps every moment), fp64
    if ((options & ACM_OPT_MOMENTS) && ((options & (ACM_OPT_INPLACE | ACM_OPT_UNFUSED | ACM_OPT_PHASE_SRT)) || precision != ACM_F64)) return false;
    const int grids = (options & ACM_OPT_INPLACE) ? 1 : 2;
    if (nx <= 0 || ny <= 0 || nz <= 0 || !valid_stencil(Qh) || !valid_stencil(Qg)) return false;
    if ((Qh == 9) != (Qg == 9)) return false;      // the two-dimensional instance uses D2Q9 for both LB steps
    if (precision != ACM_F64 && precision != ACM_F32) return false;
    const double cells = (double)nx * ny * nz;
    if (cells >= 2147483648.0) return false;
    const size_t N = (size_t)nx * ny * nz, e = precision == ACM_F64 ? 8 : 4;
    size_t o = 0;
    // planes per population set: the populations, or the coefficients of the moment representation (A, b / A, b, T)
    const bool mom = (options & ACM_OPT_MOMENTS) != 0;
    const size_t Sh = mom ? MOM_H : (size_t)Qh, Sg = mom ? MOM_G : (size_t)Qg;
    for (int b = 0; b < grids; ++b) { L->offH[b] = o; o = align256(o + Sh * N * e); }
    for (int b = 0; b < grids; ++b) { L->offG[b] = o; o = align256(o + Sg * N * e); }
    if (grids == 1) { L->offH[1] = L->offH[0]; L->offG[1] = L->offG[0]; }
    for (int b = 0; b < 2; ++b) { L->offC[b] = o; o = align256(o + N * e); }
    L->offU[0] = L->offU[1] = o; o = align256(o + 3 * N * e);
    if (options & (ACM_OPT_UNFUSED | ACM_OPT_MOMENTS)) { L->offU[1] = o; o = align256(o + 3 * N * e); }   // u double-buffered (unfused_impl.cuh, moment_impl.cuh)
    L->offStage = o; o = align256(o + 5 * N * e);
    L->offRed = o; o = align256(o + (size_t)DIAG_WIDTH * (RED_BLOCKS + 1) * sizeof(double));
    L->total = o;
    return true;
}

static int check_launch(acm_ctx* c, const char* what, cudaError_t e, int count = 1)
{
    c->launches += count;
    if (e != cudaSuccess) {
        c->sticky = ACM_ECUDA;
        return fail(ACM_ECUDA, "%s: %s", what, cudaGetErrorString(e));
    }
    return ACM_OK;
}

// Launch geometry of the two LB kernels: x-rows tiled by the block, or -- when the block is 1-D and
// nx is not a multiple of it (e.g. the paper's 260^3) -- a linear launch over all cells.
// (with two cells per thread a row has nx / 2 pairs)
static bool lb_linear(const acm_ctx* c, int cpt) { return c->block.y == 1 && c->block.z == 1 && (c->nx / cpt) % (int)c->block.x != 0; }

// geometry block of a launch over the owned planes [z0, z1) (relative to the first owned plane)
static Geom geom_of(const acm_ctx* c, bool linear, int z0, int z1)
{
    Geom g;
    g.nx = c->nx; g.ny = c->ny; g.nz = c->nz;
    g.walls = c->walls;
    g.linear = linear ? 1 : 0;
    g.zlo = c->zlo; g.zhi = c->zlo + c->nzl;
    g.zghost = c->ghost;
    g.lz0 = c->zlo + z0; g.lz1 = c->zlo + z1;
    return g;
}
static Geom geom_of(const acm_ctx* c) { return geom_of(c, false, 0, c->nzl); }

static Launch launch_over(const acm_ctx* c, dim3 b, bool linear, int nplanes, int cpt = 1)
{
    const int nxe = c->nx / cpt;      // threads along a row
    if (linear) {
        const size_t cells = (size_t)nxe * c->ny * nplanes;
        return Launch{dim3((unsigned)((cells + b.x - 1) / b.x), 1, 1), b, c->stream};
    }
    return Launch{dim3((nxe + b.x - 1) / b.x, (c->ny + b.y - 1) / b.y, (nplanes + b.z - 1) / b.z), b, c->stream};
}

static Launch lb_launch(const acm_ctx* c, int nplanes, int cpt) { return launch_over(c, c->block, lb_linear(c, cpt), nplanes, cpt); }

// Moment representation: the marching kernels (shared-memory window, moment_impl.cuh) for grids that fill the GPU, the
// direct kernels otherwise; planes per block chosen such that the blocks fill whole waves of 2 blocks per SM, counting
// the two extra planes a chunk reads.
static bool mom_march(const acm_ctx* c)
{
    if (c->nx % 2 != 0) return false;      // their loader copies aligned pairs of cells
    if (c->mom_mode >= 0) return c->mom_mode == 1;
    return c->Qh != 9 && (size_t)c->nx * c->ny * c->nzl >= ((size_t)1 << 21);
}

static int mom_zchunk(const acm_ctx* c, int planes)
{
    if (c->mom_zchunk > 0) return c->mom_zchunk < planes ? c->mom_zchunk : planes;
    const long long tiles = (long long)((c->nx + 31) / 32) * ((c->ny + 7) / 8), slots = 2LL * (c->sm_count > 0 ? c->sm_count : 148);
    int best = planes;
    double best_eff = -1.0;
    for (int zc = planes < 8 ? planes : 8; zc <= planes; ++zc) {
        const long long blocks = tiles * ((planes + zc - 1) / zc), waves = (blocks + slots - 1) / slots;
        const double eff = (double)blocks / (double)(waves * slots) * zc / (zc + 1.0);
        if (eff > best_eff + 1e-9) { best_eff = eff; best = zc; }
    }
    return best;
}

template <typename T> static T* wsp(acm_ctx* c, size_t off) { return reinterpret_cast<T*>(c->ws + off); }

// ---- typed implementations -----------------------------------------------------------------
static Launch aux_launch(const acm_ctx* c) { return launch_over(c, dim3(128, 1, 1), false, c->nzl); }

template <typename T>
static int init_t(acm_ctx* c, const void* phi, const void* u)
{
    const bool inplace = (c->options & ACM_OPT_INPLACE) != 0;
    T *H = wsp<T>(c, c->offH[0]), *G = wsp<T>(c, c->offG[0]), *C = wsp<T>(c, c->offC[0]), *U = wsp<T>(c, c->offU[0]);
    if (c->options & ACM_OPT_MOMENTS) {
        if constexpr (std::is_same<T, double>::value) {
            cudaError_t e = launch_init_mom<T>(aux_launch(c), (const T*)phi, (const T*)u, H, G, C, U, wsp<T>(c, c->offU[1]), geom_of(c), c->N);
            c->stH = ST_POST; c->stG = ST_IN;      // g: the cell's own incoming populations until the first hydrodynamic step
            c->curH = c->curG = c->curC = c->curU = c->uH = 0;
            return check_launch(c, "init_mom_kernel", e);
        } else return fail(ACM_EINVAL, "acm_init: ACM_OPT_MOMENTS is fp64 only");
    }
    cudaError_t e = launch_init<T>(c->Qh, c->Qg, inplace, aux_launch(c), (const T*)phi, (const T*)u, H, G, C, U,
                                   geom_of(c), c->N, (T)c->ref);
    if (inplace) { c->stH = ST_SWAP; c->stG = ST_IN; }
    else c->stH = c->stG = ST_POST;
    c->curH = c->curG = c->curC = c->curU = c->uH = 0;
    return check_launch(c, "init_kernel", e);
}

// state of the array after a step that read it in state s
static int next_state(int s) { return s == ST_POST ? ST_POST : (s == ST_IN ? ST_SWAP : ST_IN); }

// Peer mode: the neighbours' array at the same workspace offset, shifted by the slab height so that this slab's
// index of the plane just below (above) its owned range addresses the neighbour's last (first) owned plane.
template <typename T>
static Peers<T> peers_at(const acm_ctx* c, size_t off)
{
    if (!c->peer_on) return Peers<T>{nullptr, nullptr};
    const ptrdiff_t shift = (ptrdiff_t)c->nzl * c->nx * c->ny;
    return Peers<T>{reinterpret_cast<const T*>(c->peer_lo + off) + shift, reinterpret_cast<const T*>(c->peer_hi + off) - shift};
}

// The LB kernels can be launched on a range of owned planes [z0, z1) (inner / outer split of a slab,
// Alg. 2 lines 4-10); the buffers flip when the step is committed.
template <typename T>
static int launch_phase_range(acm_ctx* c, int z0, int z1)
{
    if (z1 <= z0) return ACM_OK;
    if (c->options & ACM_OPT_MOMENTS) {
        if constexpr (std::is_same<T, double>::value) {
            MomPhaseArgs<T> a;
            a.Msrc = wsp<T>(c, c->offH[c->curH]); a.Mdst = wsp<T>(c, c->offH[c->curH ^ 1]);
            a.Csrc = wsp<T>(c, c->offC[c->curC]); a.Cdst = wsp<T>(c, c->offC[c->curC ^ 1]);
            a.Uold = wsp<T>(c, c->offU[c->uH]); a.U = wsp<T>(c, c->offU[c->curU]);
            a.g = geom_of(c, lb_linear(c, 1), z0, z1);
            a.N = (unsigned)c->N;
            a.one_minus_omega = (T)(1.0 - 1.0 / (3.0 * c->M + 0.5));
            a.inv_xi = (T)(1.0 / c->xi);
            const bool march = mom_march(c);
            if (march) a.g = geom_of(c, false, z0, z1);
            cudaError_t e = march ? launch_phase_mom_march<T>(c->Qh, c->walls != 0, mom_zchunk(c, z1 - z0), c->stream, a)
                                  : launch_phase_mom<T>(c->Qh, c->walls != 0, lb_launch(c, z1 - z0, 1), a);
            c->phase_planes += z1 - z0;
            return check_launch(c, march ? "phase_mom_march_kernel" : "phase_mom_kernel", e);
        } else return fail(ACM_EINVAL, "ACM_OPT_MOMENTS is fp64 only");
    }
    PhaseArgs<T> a;
    a.Hsrc = wsp<T>(c, c->offH[c->curH]); a.Hdst = wsp<T>(c, c->offH[c->curH ^ 1]);
    a.Csrc = wsp<T>(c, c->offC[c->curC]); a.Cdst = wsp<T>(c, c->offC[c->curC ^ 1]);
    a.U = wsp<T>(c, c->offU[c->curU]);
    const int cpt = (c->options & ACM_OPT_UNFUSED) ? 1 : c->cpt_phase;
    a.g = geom_of(c, lb_linear(c, cpt), z0, z1);
    a.N = (unsigned)c->N;
    const double omega = 1.0 / (3.0 * c->M + 0.5);     // tau_phi = M/c_s^2 (eq. 2), shifted by 1/2
    a.one_minus_omega = (T)(1.0 - omega);
    a.inv_xi = (T)(1.0 / c->xi);
    a.ref = (T)c->ref;
    a.Hpeer = peers_at<T>(c, c->offH[c->curH]);
    a.Cpeer = peers_at<T>(c, c->offC[c->curC]);
    const Launch l = lb_launch(c, z1 - z0, cpt);
    const int coll = (c->options & ACM_OPT_PHASE_SRT) ? PHASE_SRT : PHASE_MRT;
    const bool unfused = (c->options & ACM_OPT_UNFUSED) != 0;
    cudaError_t e = unfused ? launch_unfused_phase<T>(c->Qh, c->walls != 0, coll, l, a)
                    : cpt == 2 ? launch_phase2<T>(c->Qh, c->walls != 0, c->stH, coll, l, a)
                                  : launch_phase<T>(c->Qh, c->walls != 0, c->stH, coll, l, a);
    c->phase_planes += z1 - z0;
    return check_launch(c, unfused ? "stream_h/phi/collide_h kernels" : "phase_kernel", e, unfused ? 3 : 1);
}

static void commit_phase(acm_ctx* c)
{
    c->phase_planes = 0;
    c->curH ^= 1; c->curC ^= 1;
    c->uH = c->curU;      // the velocity this phase-field step collided with
    c->stH = next_state(c->stH);
}

template <typename T>
static int launch_hydro_range(acm_ctx* c, int z0, int z1)
{
    if (z1 <= z0) return ACM_OK;
    HydroArgs<T> a;
    a.Gsrc = wsp<T>(c, c->offG[c->curG]); a.Gdst = wsp<T>(c, c->offG[c->curG ^ 1]);
    a.C = wsp<T>(c, c->offC[c->curC]);
    a.U = wsp<T>(c, c->offU[c->curU]);
    const int cpt = (c->options & ACM_OPT_UNFUSED) ? 1 : c->cpt_hydro;
    a.g = geom_of(c, lb_linear(c, cpt), z0, z1);
    a.N = (unsigned)c->N;
    // rho and tau at the reference phase of the stored phi (ref = 0: the light phase, as in eqs. 8, 20)
    a.ref = (T)c->ref;
    a.rho_L = (T)(c->rho_L + c->ref * (c->rho_H - c->rho_L)); a.drho = (T)(c->rho_H - c->rho_L);
    a.tau_L = (T)(3.0 * c->nu_L + c->ref * (3.0 * c->nu_H - 3.0 * c->nu_L)); a.dtau = (T)(3.0 * c->nu_H - 3.0 * c->nu_L);
    a.beta4 = (T)(4.0 * 12.0 * c->sigma / c->xi); a.kappa = (T)(1.5 * c->sigma * c->xi);
    a.gx = (T)c->grav[0]; a.gy = (T)c->grav[1]; a.gz = (T)c->grav[2];
    a.bulk_one = (c->options & ACM_OPT_BULK_ONE) ? 1 : 0;
    a.subiter = c->subiter;
    a.Gpeer = peers_at<T>(c, c->offG[c->curG]);
    a.Cpeer = peers_at<T>(c, c->offC[c->curC]);
    if (c->options & ACM_OPT_MOMENTS) {
        if constexpr (std::is_same<T, double>::value) {
            MomHydroArgs<T> ma;
            ma.h = a;
            ma.h.g = geom_of(c, lb_linear(c, 1), z0, z1);
            ma.Ksrc = wsp<T>(c, c->offG[c->curG]); ma.Kdst = wsp<T>(c, c->offG[c->curG ^ 1]);
            ma.Uin = wsp<T>(c, c->offU[c->curU]); ma.Uout = wsp<T>(c, c->offU[c->curU ^ 1]);
            const bool march = mom_march(c) && c->stG != ST_IN;      // the first step after acm_init (no streaming) stays direct
            if (march) ma.h.g = geom_of(c, false, z0, z1);
            cudaError_t e = march ? launch_hydro_mom_march<T>(c->Qg, c->walls != 0, mom_zchunk(c, z1 - z0), c->stream, ma)
                                  : launch_hydro_mom<T>(c->Qg, c->walls != 0, c->stG == ST_IN, lb_launch(c, z1 - z0, 1), ma);
            c->hydro_planes += z1 - z0;
            return check_launch(c, march ? "hydro_mom_march_kernel" : "hydro_mom_kernel", e);
        } else return fail(ACM_EINVAL, "ACM_OPT_MOMENTS is fp64 only");
    }
    const Launch l = lb_launch(c, z1 - z0, cpt);
    const bool unfused = (c->options & ACM_OPT_UNFUSED) != 0;
    cudaError_t e = unfused ? launch_unfused_hydro<T>(c->Qg, c->walls != 0, l, a, wsp<T>(c, c->offU[c->curU]), wsp<T>(c, c->offU[c->curU ^ 1]))
                    : cpt == 2 ? launch_hydro2<T>(c->Qg, c->walls != 0, c->stG, l, a)
                                  : launch_hydro<T>(c->Qg, c->walls != 0, c->stG, l, a);
    c->hydro_planes += z1 - z0;
    return check_launch(c, unfused ? "stream_g/velocity/collide_g kernels" : "hydro_kernel", e, unfused ? 3 : 1);
}

static void commit_hydro(acm_ctx* c)
{
    c->hydro_planes = 0;
    c->steps_done += 1;
    if (c->options & (ACM_OPT_UNFUSED | ACM_OPT_MOMENTS)) c->curU ^= 1;
    c->curG ^= 1;
    c->stG = (c->options & ACM_OPT_MOMENTS) ? ST_POST : next_state(c->stG);
}

template <typename T>
static int launch_phase_step(acm_ctx* c)
{
    int rc = launch_phase_range<T>(c, 0, c->nzl);
    if (rc == ACM_OK) commit_phase(c);
    return rc;
}

template <typename T>
static int launch_hydro_step(acm_ctx* c)
{
    int rc = launch_hydro_range<T>(c, 0, c->nzl);
    if (rc == ACM_OK) commit_hydro(c);
    return rc;
}

static void prof_mark(acm_ctx* c)
{
    if (!c->profiling || c->ev_used >= c->ev.size()) return;
    cudaEventRecord(c->ev[c->ev_used++], c->stream);
}

// make sure the pool holds `count` unused events (created here, outside the kernel sequence)
static bool prof_reserve(acm_ctx* c, size_t count)
{
    while (c->ev.size() < c->ev_used + count) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return false;
        c->ev.push_back(e);
    }
    return true;
}

static void graphs_clear(acm_ctx* c)
{
    for (auto& g : c->graphs) cudaGraphExecDestroy(g.exec);
    c->graphs.clear();
}

static unsigned graph_key(const acm_ctx* c)
{
    return (unsigned)c->curH | (unsigned)c->curG << 1 | (unsigned)c->curC << 2 | (unsigned)c->curU << 3 | (unsigned)c->stH << 4 | (unsigned)c->stG << 6 | (unsigned)c->uH << 8;
}

static bool graph_wanted(const acm_ctx* c)
{
    if (c->profiling || c->ghost) return false;
    return c->graph_mode > 0 || (c->graph_mode < 0 && (size_t)c->nx * c->ny * c->nzl <= GRAPH_AUTO_CELLS);
}

template <typename T> static int plain_steps(acm_ctx* c, int n);

// the executable graph of GRAPH_STEPS steps starting from the current buffer parity (captured on first use)
template <typename T>
static cudaGraphExec_t graph_for_state(acm_ctx* c)
{
    const unsigned key = graph_key(c);
    for (auto& g : c->graphs)
        if (g.key == key) return g.exec;
    if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    const cudaStream_t user = c->stream;
    const long long launches = c->launches, steps_done = c->steps_done;
    const int stG = c->stG, uH = c->uH;      // moment representation: these two do not come back after an even count
    c->stream = c->cap_stream;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    bool ok = cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) {
        ok = plain_steps<T>(c, GRAPH_STEPS) == ACM_OK;      // recorded, not executed; the state is back where it was (even count)
        ok = (cudaStreamEndCapture(c->cap_stream, &graph) == cudaSuccess) && ok && graph;
    }
    if (ok) ok = cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess;
    if (graph) cudaGraphDestroy(graph);
    c->stream = user;
    c->launches = launches;
    c->steps_done = steps_done;
    c->stG = stG; c->uH = uH;
    if (!ok) {
        cudaGetLastError();
        c->sticky = ACM_OK;          // a failed capture is not a failed launch: fall back to plain launches
        c->graph_mode = 0;
        return nullptr;
    }
    c->graphs.push_back({key, exec});
    return exec;
}

template <typename T>
static int plain_steps(acm_ctx* c, int n)
{
    for (int t = 0; t < n; ++t) {
        int rc = launch_phase_step<T>(c);
        if (rc) return rc;
        prof_mark(c);
        rc = launch_hydro_step<T>(c);
        if (rc) return rc;
        prof_mark(c);
    }
    return ACM_OK;
}

template <typename T>
static int step_t(acm_ctx* c, int n)
{
    if (c->profiling && n > 0) {
        if (!prof_reserve(c, 2 * (size_t)n + 1)) return fail(ACM_ECUDA, "acm_step: cudaEventCreate failed");
        c->ev_calls.push_back(n);
        prof_mark(c);
    }
    int done = 0;
    if (graph_wanted(c)) {
        const int per_step = (c->options & ACM_OPT_UNFUSED) ? 6 : 2;
        while (n - done >= GRAPH_STEPS) {
            cudaGraphExec_t exec = graph_for_state<T>(c);
            if (!exec) break;
            cudaError_t e = cudaGraphLaunch(exec, c->stream);
            if (e != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "acm_step: cudaGraphLaunch: %s", cudaGetErrorString(e)); }
            c->launches += (long long)per_step * GRAPH_STEPS;
            c->steps_done += GRAPH_STEPS;
            c->graph_replays += 1;
            done += GRAPH_STEPS;
            if (c->options & ACM_OPT_MOMENTS) { c->stG = ST_POST; c->uH = c->curU ^ 1; }      // the state any completed step leaves
        }
    }
    return plain_steps<T>(c, n - done);
}

template <typename T>
static int export_g_t(acm_ctx* c, void* g, void* p)      // incoming convention (+ pressure)
{
    if (c->options & ACM_OPT_MOMENTS) {
        if constexpr (std::is_same<T, double>::value) {
            cudaError_t e = launch_export_g_mom<T>(c->Qg, c->stG == ST_IN, aux_launch(c), wsp<T>(c, c->offG[c->curG]), wsp<T>(c, c->offC[c->curC]),
                                                   (T*)g, (T*)p, geom_of(c), c->N, (T)c->rho_L, (T)(c->rho_H - c->rho_L));
            return check_launch(c, "export_g_mom_kernel", e);
        } else return fail(ACM_EINVAL, "ACM_OPT_MOMENTS is fp64 only");
    }
    cudaError_t e = launch_export<T>(c->Qg, c->stG, false, aux_launch(c), wsp<T>(c, c->offG[c->curG]), wsp<T>(c, c->offC[c->curC]),
                                     (T*)g, (T*)p, geom_of(c), c->N, (T)(c->rho_L + c->ref * (c->rho_H - c->rho_L)), (T)(c->rho_H - c->rho_L), (T)0);
    return check_launch(c, "export_kernel", e);
}

template <typename T>
static int export_h_t(acm_ctx* c, void* h)               // post-collision convention
{
    if (c->options & ACM_OPT_MOMENTS) {
        if constexpr (std::is_same<T, double>::value) {
            cudaError_t e = launch_export_h_mom<T>(c->Qh, aux_launch(c), wsp<T>(c, c->offH[c->curH]), wsp<T>(c, c->offC[c->curC]),
                                                   wsp<T>(c, c->offU[c->uH]), (T*)h, geom_of(c), c->N);
            return check_launch(c, "export_h_mom_kernel", e);
        } else return fail(ACM_EINVAL, "ACM_OPT_MOMENTS is fp64 only");
    }
    cudaError_t e = launch_export<T>(c->Qh, c->stH, true, aux_launch(c), wsp<T>(c, c->offH[c->curH]), wsp<T>(c, c->offC[c->curC]),
                                     (T*)h, (T*)nullptr, geom_of(c), c->N, (T)c->rho_L, (T)(c->rho_H - c->rho_L), (T)c->ref);
    return check_launch(c, "export_kernel", e);
}

template <typename T>
static int import_g_t(acm_ctx* c, const void* g)      // incoming convention -> ST_POST storage
{
    cudaError_t e = launch_import<T>(c->Qg, false, aux_launch(c), (const T*)g, wsp<T>(c, c->offG[c->curG]),
                                     geom_of(c), c->N, (T)0);
    return check_launch(c, "import_kernel", e);
}

template <typename T>
static int import_h_t(acm_ctx* c, const void* h)      // post-collision convention -> ST_SWAP storage
{
    cudaError_t e = launch_import<T>(c->Qh, true, aux_launch(c), (const T*)h, wsp<T>(c, c->offH[c->curH]),
                                     geom_of(c), c->N, (T)c->ref);
    return check_launch(c, "import_kernel", e);
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

// dst = phi-field-like source + shift (device to device); a plain copy when shift = 0
static int copy_field_shifted(acm_ctx* c, void* dst, const void* src, size_t n, double shift, const char* what)
{
    if (shift == 0.0) return copy_async(c, dst, src, n * c->esz, cudaMemcpyDeviceToDevice, what);
    cudaError_t e = c->precision == ACM_F64 ? launch_shift_field<double>(c->stream, (const double*)src, (double*)dst, n, shift)
                                            : launch_shift_field<float>(c->stream, (const float*)src, (float*)dst, n, (float)shift);
    return check_launch(c, what, e);
}

#define ACM_CHECK_CTX(c)                                                          \
    if (!(c)) return fail(ACM_EINVAL, "%s: NULL context", __func__);              \
    if ((c)->sticky) return fail(ACM_ECUDA, "%s: context has a sticky CUDA error", __func__)

// Default cells per thread and block.  fp32: two cells per thread (8-byte accesses, packed fp32 arithmetic) whenever
// the rows allow it.  fp64: the pairing (16-byte accesses) saves index arithmetic, hence power: +1.8 % at D3Q15 / D3Q19
// under the sustained 1 kW power cap, nothing in a burst, while the 250 registers of a D3Q27 pair cost 2-5 % and the
// D2Q9 hydrodynamic pair 6 % (profiles/r2_profiles.md) -- so two cells for the phase kernel up to D3Q19 and for the
// hydrodynamic kernel at D3Q15 / D3Q19, one otherwise.
// One block = 1 KB of every population row (measured best on B200 for both precisions, profiles/): 128 fp64 cells or
// 256 fp32 cells (128 pairs) along x; single-cell fp32 falls back to 128 when nx is not a multiple of 256.
static void default_cells_per_thread(acm_ctx* c)
{
    const bool can_pair = c->nx % 2 == 0 && !(c->options & (ACM_OPT_UNFUSED | ACM_OPT_MOMENTS));
    const bool f32 = c->precision == ACM_F32;
    c->cpt_phase = (can_pair && (f32 || c->Qh <= 19)) ? 2 : 1;
    c->cpt_hydro = (can_pair && (f32 || c->Qg == 15 || c->Qg == 19)) ? 2 : 1;
    c->block = (f32 && c->cpt_phase == 1 && c->nx % 256 == 0) ? dim3(256, 1, 1) : dim3(128, 1, 1);
}

// nz = owned planes; rank/nranks/nz_global/zglob0 describe the slab (nranks = 0: a plain context without ghost planes)
static int create_impl(acm_ctx** out, int nx, int ny, int nz, int stencil_phase, int stencil_hydro, double rho_H, double rho_L,
                       double sigma, double xi, double M, double nu_H, double nu_L, const double gravity[3], unsigned wall_flags,
                       int precision, unsigned options, void* workspace, void* cuda_stream, int rank, int nranks, int nz_global,
                       int zglob0)
{
    const bool slab = nranks > 0;
    const int nzl = nz;
    if ((options & ACM_OPT_BULK_ONE) && (options & ACM_OPT_UNFUSED))
        return fail(ACM_EINVAL, "acm_create: ACM_OPT_BULK_ONE is not available with ACM_OPT_UNFUSED");
    if (slab) {
        if (options & (ACM_OPT_INPLACE | ACM_OPT_UNFUSED | ACM_OPT_BULK_ONE | ACM_OPT_MOMENTS))
            return fail(ACM_EINVAL, "acm_create_slab: ACM_OPT_INPLACE / ACM_OPT_UNFUSED / ACM_OPT_BULK_ONE / ACM_OPT_MOMENTS are not available for slabs");
        if (nz > 0) nz += 2;      // ghost planes below and above
    }
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
    if (stencil_phase == 9 && (nzl != 1 || slab || (gravity && gravity[2] != 0.0)))
        return fail(ACM_EINVAL, "acm_create: D2Q9 needs nz = 1, no slab decomposition and gravity[2] = 0");
    if (!workspace) return fail(ACM_EINVAL, "acm_create: workspace is NULL");
    if ((uintptr_t)workspace & 255) return fail(ACM_EINVAL, "acm_create: workspace must be 256-byte aligned");
    acm_ctx* c = new (std::nothrow) acm_ctx();
    if (!c) return fail(ACM_EINVAL, "acm_create: out of host memory");
    c->nx = nx; c->ny = ny; c->nz = nz; c->Qh = stencil_phase; c->Qg = stencil_hydro; c->precision = precision;
    c->N = (size_t)nx * ny * nz; c->esz = precision == ACM_F64 ? 8 : 4;
    c->rho_H = rho_H; c->rho_L = rho_L; c->sigma = sigma; c->xi = xi; c->M = M; c->nu_H = nu_H; c->nu_L = nu_L;
    for (int a = 0; a < 3; ++a) c->grav[a] = gravity ? gravity[a] : 0.0;
    // internal wall bits: the z walls per face; a slab has a z wall only on an outer face of the domain
    c->walls = wall_flags & (ACM_WALL_X | ACM_WALL_Y);
    if (wall_flags & ACM_WALL_Z) {
        if (!slab || rank == 0) c->walls |= WALL_ZLO;
        if (!slab || rank == nranks - 1) c->walls |= WALL_ZHI;
    }
    c->ref_mode = -1; c->ref = 0.0;
    c->peer_on = false; c->peer_lo = c->peer_hi = nullptr;
    c->nzl = nzl; c->zlo = slab ? 1 : 0; c->ghost = slab ? 1 : 0;
    c->zglob0 = zglob0; c->nz_global = slab ? nz_global : nzl; c->rank = slab ? rank : 0; c->nranks = slab ? nranks : 1;
    c->stream = (cudaStream_t)cuda_stream;
    c->ws = (char*)workspace;
    for (int b = 0; b < 2; ++b) { c->offH[b] = L.offH[b]; c->offG[b] = L.offG[b]; c->offC[b] = L.offC[b]; }
    c->offU[0] = L.offU[0]; c->offU[1] = L.offU[1]; c->offStage = L.offStage; c->offRed = L.offRed;
    c->curH = c->curG = c->curC = c->curU = 0;
    c->options = options;
    c->stH = c->stG = ST_POST;
    c->initialised = false;
    c->sticky = ACM_OK;
    default_cells_per_thread(c);
    c->launches = 0;
    c->steps_done = 0;
    c->subiter = 1;
    c->uH = 0; c->mom_mode = -1; c->mom_zchunk = 0;
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); sms = 0; }
        c->sm_count = sms;
    }
    c->phase_planes = c->hydro_planes = 0;
    c->profiling = false;
    c->ev_used = 0;
    c->graph_mode = -1;
    c->cap_stream = nullptr;
    c->graph_replays = 0;
    c->io_stream = nullptr;
    for (auto& e : c->io_ev) e = nullptr;
    *out = c;
    return ACM_OK;
}


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
    return create_impl(out, nx, ny, nz, stencil_phase, stencil_hydro, rho_H, rho_L, sigma, xi, M, nu_H, nu_L, gravity, wall_flags,
                       precision, options, workspace, cuda_stream, 0, 0, nz, 0);
}

// ---- slab decomposition along z --------------------------------------------------------------
int acm_slab_range(int nz_global, int rank, int nranks, int* z_begin, int* z_count)
{
    if (nz_global < 1 || nranks < 1 || rank < 0 || rank >= nranks || nranks > nz_global)
        return fail(ACM_EINVAL, "acm_slab_range: need 1 <= nranks <= nz_global and 0 <= rank < nranks");
    const int base = nz_global / nranks, rem = nz_global % nranks;     // the first `rem` slabs get one more plane
    if (z_begin) *z_begin = rank * base + (rank < rem ? rank : rem);
    if (z_count) *z_count = base + (rank < rem ? 1 : 0);
    return ACM_OK;
}

size_t acm_workspace_bytes_slab(int nx, int ny, int nz_global, int stencil_phase, int stencil_hydro, int precision, int rank,
                                int nranks)
{
    int z0, cnt;
    if (acm_slab_range(nz_global, rank, nranks, &z0, &cnt) != ACM_OK) return 0;
    return acm_workspace_bytes_opt(nx, ny, cnt + 2, stencil_phase, stencil_hydro, precision, 0u);
}

int acm_create_slab(acm_ctx** out, int nx, int ny, int nz_global, int stencil_phase, int stencil_hydro, double rho_H,
                    double rho_L, double sigma, double xi, double M, double nu_H, double nu_L, const double gravity[3],
                    unsigned wall_flags, int precision, unsigned options, int rank, int nranks, void* workspace,
                    void* cuda_stream)
{
    if (out) *out = nullptr;
    int z0, cnt;
    int rc = acm_slab_range(nz_global, rank, nranks, &z0, &cnt);
    if (rc) return rc;
    return create_impl(out, nx, ny, cnt, stencil_phase, stencil_hydro, rho_H, rho_L, sigma, xi, M, nu_H, nu_L, gravity, wall_flags,
                       precision, options, workspace, cuda_stream, rank, nranks, nz_global, z0);
}

int acm_slab_info(const acm_ctx* c, int info[6])
{
    if (!c || !info) return fail(ACM_EINVAL, "acm_slab_info: NULL argument");
    info[0] = c->rank; info[1] = c->nranks; info[2] = c->zglob0; info[3] = c->nzl; info[4] = c->nz; info[5] = c->ghost;
    return ACM_OK;
}

// planes that cross a z face: directions with e_z = +1 (sign > 0) or e_z = -1 (sign < 0), increasing index
static int crossing_dirs(int Q, int sign, int* dirs)
{
    int n = 0;
    for (int i = 0; i < Q; ++i) {
        const int k = (Q == 15 && i >= 7) ? i + 12 : (Q == 9 && i >= 5) ? i + 2 : i;
        if (acm::dir27(k, 2) == sign) dirs[n++] = i;
    }
    return n;
}

int acm_halo_plan(const acm_ctx* c, int what, int side, int recv, int max_chunks, size_t* offsets, size_t* bytes)
{
    if (!c || !offsets || !bytes) return -fail(ACM_EINVAL, "acm_halo_plan: NULL argument");
    if (!c->ghost) return -fail(ACM_ESTATE, "acm_halo_plan: not a slab context");
    if ((what != ACM_HALO_H && what != ACM_HALO_G && what != ACM_HALO_PHI) || (side != 0 && side != 1))
        return -fail(ACM_EINVAL, "acm_halo_plan: bad what/side");
    const size_t plane = (size_t)c->nx * c->ny * c->esz;
    // side 0 = low z face: my first owned plane (zlo) goes out, my low ghost plane (zlo-1) comes in;
    // side 1 = high z face: my last owned plane goes out, my high ghost plane comes in
    const int zplane = side == 0 ? (recv ? c->zlo - 1 : c->zlo) : (recv ? c->zlo + c->nzl : c->zlo + c->nzl - 1);
    int n = 0;
    if (what == ACM_HALO_PHI) {
        if (max_chunks < 1) return -fail(ACM_EINVAL, "acm_halo_plan: max_chunks too small");
        offsets[0] = c->offC[c->curC] + (size_t)zplane * plane;
        bytes[0] = plane;
        return 1;
    }
    // Populations are stored post-collision at their own cell and pulled by the next step: the cell at z
    // pulls slot i from z - e_iz.  My low ghost plane must hold the slots with e_z = +1 (pulled upwards into my
    // first plane); what I send through the low face fills the low neighbour's HIGH ghost: slots with e_z = -1.
    const int Q = what == ACM_HALO_H ? c->Qh : c->Qg;
    const size_t base = what == ACM_HALO_H ? c->offH[c->curH] : c->offG[c->curG];
    const int sign = (side == 0) == (recv != 0) ? +1 : -1;
    int dirs[27];
    n = crossing_dirs(Q, sign, dirs);
    if (n > max_chunks) return -fail(ACM_EINVAL, "acm_halo_plan: max_chunks too small (need %d)", n);
    for (int k = 0; k < n; ++k) {
        offsets[k] = base + ((size_t)dirs[k] * c->N) * c->esz + (size_t)zplane * plane;
        bytes[k] = plane;
    }
    return n;
}

int acm_set_peers(acm_ctx* c, void* lo_workspace, void* hi_workspace)
{
    ACM_CHECK_CTX(c);
    if (!c->ghost) return fail(ACM_ESTATE, "acm_set_peers: not a slab context");
    if (!lo_workspace && !hi_workspace) { c->peer_on = false; c->peer_lo = c->peer_hi = nullptr; return ACM_OK; }
    if (c->nz_global % c->nranks != 0) return fail(ACM_EINVAL, "acm_set_peers: needs slabs of equal height (nz_global %% nranks == 0)");
    const bool need_lo = !((c->walls & WALL_ZLO) != 0), need_hi = !((c->walls & WALL_ZHI) != 0);
    if ((need_lo && !lo_workspace) || (need_hi && !hi_workspace))
        return fail(ACM_EINVAL, "acm_set_peers: a neighbour workspace is missing on a face that is not a wall");
    // a face on a wall of the global domain has no neighbour; its pointer is never dereferenced
    c->peer_lo = lo_workspace ? (char*)lo_workspace : c->ws;
    c->peer_hi = hi_workspace ? (char*)hi_workspace : c->ws;
    c->peer_on = true;
    return ACM_OK;
}

int acm_state_signature(const acm_ctx* c, unsigned long long out[8])
{
    if (!c || !out) return fail(ACM_EINVAL, "acm_state_signature: NULL argument");
    out[0] = c->offRed + align256((size_t)DIAG_WIDTH * (RED_BLOCKS + 1) * sizeof(double));      // workspace bytes (layout total)
    out[1] = c->offH[c->curH]; out[2] = c->offG[c->curG]; out[3] = c->offC[c->curC];
    out[4] = (unsigned long long)c->steps_done;
    out[5] = (unsigned long long)c->nzl;
    out[6] = (unsigned long long)(c->phase_planes != 0 || c->hydro_planes != 0);
    out[7] = (unsigned long long)(c->precision == ACM_F32 ? (c->ref != 0.0 ? 2 : 1) : 0);
    return ACM_OK;
}

int acm_phase_launch(acm_ctx* c, int z0, int z1)
{
    ACM_CHECK_CTX(c);
    if (!c->initialised) return fail(ACM_ESTATE, "acm_phase_launch: call acm_init first");
    if (z0 < 0 || z1 > c->nzl || z0 > z1) return fail(ACM_EINVAL, "acm_phase_launch: need 0 <= z0 <= z1 <= owned planes");
    if (c->options & ACM_OPT_MOMENTS) return fail(ACM_ESTATE, "acm_phase_launch: not available with ACM_OPT_MOMENTS (use acm_step)");
    if (c->phase_planes + (z1 - z0) > c->nzl) return fail(ACM_ESTATE, "acm_phase_launch: more planes than the slab owns since the last acm_phase_commit");
    if (c->hydro_planes) return fail(ACM_ESTATE, "acm_phase_launch: the hydrodynamic step is not committed");
    return c->precision == ACM_F64 ? launch_phase_range<double>(c, z0, z1) : launch_phase_range<float>(c, z0, z1);
}

int acm_phase_commit(acm_ctx* c)
{
    ACM_CHECK_CTX(c);
    if (c->phase_planes != c->nzl)
        return fail(ACM_ESTATE, "acm_phase_commit: %d of %d owned planes were launched since the last commit", c->phase_planes, c->nzl);
    commit_phase(c);
    return ACM_OK;
}

int acm_hydro_launch(acm_ctx* c, int z0, int z1)
{
    ACM_CHECK_CTX(c);
    if (!c->initialised) return fail(ACM_ESTATE, "acm_hydro_launch: call acm_init first");
    if (z0 < 0 || z1 > c->nzl || z0 > z1) return fail(ACM_EINVAL, "acm_hydro_launch: need 0 <= z0 <= z1 <= owned planes");
    if (c->options & ACM_OPT_MOMENTS) return fail(ACM_ESTATE, "acm_hydro_launch: not available with ACM_OPT_MOMENTS (use acm_step)");
    if (c->hydro_planes + (z1 - z0) > c->nzl) return fail(ACM_ESTATE, "acm_hydro_launch: more planes than the slab owns since the last acm_hydro_commit");
    if (c->phase_planes) return fail(ACM_ESTATE, "acm_hydro_launch: the phase-field step is not committed");
    return c->precision == ACM_F64 ? launch_hydro_range<double>(c, z0, z1) : launch_hydro_range<float>(c, z0, z1);
}

int acm_hydro_commit(acm_ctx* c)
{
    ACM_CHECK_CTX(c);
    if (c->hydro_planes != c->nzl)
        return fail(ACM_ESTATE, "acm_hydro_commit: %d of %d owned planes were launched since the last commit", c->hydro_planes, c->nzl);
    commit_hydro(c);
    return ACM_OK;
}

static void prof_clear(acm_ctx* c)      // forget the records, keep the pool
{
    c->ev_used = 0;
    c->ev_calls.clear();
}

void acm_destroy(acm_ctx* c)
{
    if (!c) return;
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    graphs_clear(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->io_stream) cudaStreamDestroy(c->io_stream);
    for (cudaEvent_t e : c->io_ev) if (e) cudaEventDestroy(e);
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
        if (k + 2 * (size_t)n + 1 > c->ev_used) break;
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
    if (c->phase_planes || c->hydro_planes) return fail(ACM_ESTATE, "acm_set_block: a step is partly launched (commit it first)");
    c->block = dim3(bx, by, bz);
    graphs_clear(c);
    return ACM_OK;
}

int acm_set_cells_per_thread(acm_ctx* c, int phase, int hydro)
{
    ACM_CHECK_CTX(c);
    if (phase < 0 || phase > 2 || hydro < 0 || hydro > 2) return fail(ACM_EINVAL, "acm_set_cells_per_thread: 0 (default), 1 or 2");
    if ((phase == 2 || hydro == 2) && (c->nx % 2 != 0 || (c->options & (ACM_OPT_UNFUSED | ACM_OPT_MOMENTS))))
        return fail(ACM_EINVAL, "acm_set_cells_per_thread: two cells per thread need an even nx and the fused kernels");
    if (c->phase_planes || c->hydro_planes) return fail(ACM_ESTATE, "acm_set_cells_per_thread: a step is partly launched (commit it first)");
    const dim3 block = c->block;
    default_cells_per_thread(c);
    c->block = block;
    if (phase) c->cpt_phase = phase;
    if (hydro) c->cpt_hydro = hydro;
    graphs_clear(c);
    return ACM_OK;
}

int acm_set_subiter(acm_ctx* c, int sweeps)
{
    ACM_CHECK_CTX(c);
    if (sweeps < 1 || sweeps > 64) return fail(ACM_EINVAL, "acm_set_subiter: need 1 <= sweeps <= 64");
    if (sweeps > 1 && (c->ghost || (c->options & ACM_OPT_UNFUSED)))
        return fail(ACM_EINVAL, "acm_set_subiter: not available for slabs or with ACM_OPT_UNFUSED");
    if (c->phase_planes || c->hydro_planes) return fail(ACM_ESTATE, "acm_set_subiter: a step is partly launched (commit it first)");
    c->subiter = sweeps;
    graphs_clear(c);
    return ACM_OK;
}

int acm_set_moment_kernels(acm_ctx* c, int mode, int zchunk)
{
    ACM_CHECK_CTX(c);
    if (!(c->options & ACM_OPT_MOMENTS)) return fail(ACM_ESTATE, "acm_set_moment_kernels: the context was not created with ACM_OPT_MOMENTS");
    if (mode < -1 || mode > 1 || zchunk < 0) return fail(ACM_EINVAL, "acm_set_moment_kernels: mode must be -1, 0 or 1 and zchunk >= 0");
    c->mom_mode = mode; c->mom_zchunk = zchunk;
    graphs_clear(c);
    return ACM_OK;
}

int acm_set_graph(acm_ctx* c, int mode)
{
    ACM_CHECK_CTX(c);
    if (mode < -1 || mode > 1) return fail(ACM_EINVAL, "acm_set_graph: mode must be -1 (automatic), 0 (never) or 1 (always)");
    c->graph_mode = mode;
    return ACM_OK;
}

long long acm_graph_replays(const acm_ctx* c) { return c ? c->graph_replays : 0; }

long long acm_launch_count(const acm_ctx* c) { return c ? c->launches : 0; }

int acm_init(acm_ctx* c, const void* phi, const void* u)
{
    ACM_CHECK_CTX(c);
    if (!phi || !u) return fail(ACM_EINVAL, "acm_init: phi and u are required");
    graphs_clear(c);                  // the reference phase of the fp32 instance is a kernel argument
    c->phase_planes = c->hydro_planes = 0;
    c->steps_done = 0;
    c->ref = 0.0;
    if (c->precision == ACM_F32) {
        // reference phase of the deviation storage: the phase that fills most of the domain
        if (c->ref_mode >= 0) c->ref = c->ref_mode;
        else if (c->ghost) c->ref = 1.0;      // every slab of a decomposition must take the same one: bubbles in liquid
        else {
            double* part = wsp<double>(c, c->offRed);
            double total = 0.0;
            int rc0 = check_launch(c, "sum_phi", launch_sum_phi<float>(c->stream, (const float*)phi, c->N, part), 2);
            if (!rc0) rc0 = copy_async(c, &total, part + RED_BLOCKS, sizeof(double), cudaMemcpyDeviceToHost, "acm_init(mean phi)");
            if (rc0) return rc0;
            if (cudaStreamSynchronize(c->stream) != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "acm_init: synchronize failed"); }
            c->ref = total > 0.5 * (double)c->N ? 1.0 : 0.0;
        }
    }
    int rc = c->precision == ACM_F64 ? init_t<double>(c, phi, u) : init_t<float>(c, phi, u);
    if (rc == ACM_OK && c->ghost) {
        // slab: phi and u come with their ghost planes filled (the pre-shifted g needs u of the neighbour planes);
        // the phi ghost planes are taken over as they are, those of h and g arrive with the first halo exchange
        const size_t plane = (size_t)c->nx * c->ny * c->esz;
        const size_t hi = (size_t)(c->zlo + c->nzl) * plane;
        const size_t cells = (size_t)c->nx * c->ny;
        rc = copy_field_shifted(c, c->ws + c->offC[0], phi, cells, -c->ref, "acm_init(phi ghost)");
        if (!rc) rc = copy_field_shifted(c, c->ws + c->offC[0] + hi, (const char*)phi + hi, cells, -c->ref, "acm_init(phi ghost)");
    }
    if (rc == ACM_OK) c->initialised = true;
    return rc;
}

int acm_set_reference_phase(acm_ctx* c, int phase)
{
    ACM_CHECK_CTX(c);
    if (phase < -1 || phase > 1) return fail(ACM_EINVAL, "acm_set_reference_phase: phase must be -1 (automatic), 0 (light) or 1 (heavy)");
    if (c->initialised) return fail(ACM_ESTATE, "acm_set_reference_phase: must be called before acm_init");
    c->ref_mode = phase;
    return ACM_OK;
}

int acm_step(acm_ctx* c, int n)
{
    ACM_CHECK_CTX(c);
    if (n < 0) return fail(ACM_EINVAL, "acm_step: n must be >= 0");
    if (!c->initialised) return fail(ACM_ESTATE, "acm_step: call acm_init first");
    if (c->ghost && n > 0) return fail(ACM_ESTATE, "acm_step: a slab advances with acm_phase_launch / acm_hydro_launch and the halo exchange");
    return c->precision == ACM_F64 ? step_t<double>(c, n) : step_t<float>(c, n);
}

int acm_fields(acm_ctx* c, void* phi, void* u, void* p)
{
    ACM_CHECK_CTX(c);
    if (!c->initialised) return fail(ACM_ESTATE, "acm_fields: call acm_init first");
    int rc = ACM_OK;
    if (phi) rc = copy_field_shifted(c, phi, c->ws + c->offC[c->curC], c->N, c->ref, "acm_fields(phi)");
    if (!rc && u) rc = copy_async(c, u, c->ws + c->offU[c->curU], 3 * c->N * c->esz, cudaMemcpyDeviceToDevice, "acm_fields(u)");
    if (!rc && p) rc = c->precision == ACM_F64 ? export_g_t<double>(c, nullptr, p) : export_g_t<float>(c, nullptr, p);
    return rc;
}

int acm_phi_mass(acm_ctx* c, double* total_host)
{
    ACM_CHECK_CTX(c);
    if (!total_host) return fail(ACM_EINVAL, "acm_phi_mass: total_host is NULL");
    if (!c->initialised) return fail(ACM_ESTATE, "acm_phi_mass: call acm_init first");
    double* part = wsp<double>(c, c->offRed);
    const size_t first = (size_t)c->zlo * c->nx * c->ny, owned = (size_t)c->nzl * c->nx * c->ny;   // a slab sums its own planes
    cudaError_t le = c->precision == ACM_F64 ? launch_sum_phi<double>(c->stream, wsp<double>(c, c->offC[c->curC]) + first, owned, part)
                                             : launch_sum_phi<float>(c->stream, wsp<float>(c, c->offC[c->curC]) + first, owned, part);
    int rc = check_launch(c, "sum_phi", le, 2);
    if (rc) return rc;
    rc = copy_async(c, total_host, part + RED_BLOCKS, sizeof(double), cudaMemcpyDeviceToHost, "acm_phi_mass");
    if (rc) return rc;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "acm_phi_mass: %s", cudaGetErrorString(e)); }
    *total_host += c->ref * (double)owned;        // fp32 instance: the field holds phi - ref
    if (!std::isfinite(*total_host)) return fail(ACM_EUNSTABLE, "acm_phi_mass: sum(phi) is not finite");
    return ACM_OK;
}

int acm_bubble_sums(acm_ctx* c, double out_host[7])
{
    ACM_CHECK_CTX(c);
    if (!out_host) return fail(ACM_EINVAL, "acm_bubble_sums: out_host is NULL");
    if (!c->initialised) return fail(ACM_ESTATE, "acm_bubble_sums: call acm_init first");
    double* part = wsp<double>(c, c->offRed);
    const Geom g = geom_of(c);
    const int zshift = c->zglob0 - c->zlo;
    cudaError_t le = c->precision == ACM_F64
                         ? launch_bubble_diag<double>(c->stream, wsp<double>(c, c->offC[c->curC]), wsp<double>(c, c->offU[c->curU]), g, c->N, zshift, c->ref, part)
                         : launch_bubble_diag<float>(c->stream, wsp<float>(c, c->offC[c->curC]), wsp<float>(c, c->offU[c->curU]), g, c->N, zshift, c->ref, part);
    int rc = check_launch(c, "bubble_diag", le, 2);
    if (rc) return rc;
    rc = copy_async(c, out_host, part + (size_t)DIAG_WIDTH * RED_BLOCKS, DIAG_WIDTH * sizeof(double), cudaMemcpyDeviceToHost, "acm_bubble_sums");
    if (rc) return rc;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "acm_bubble_sums: %s", cudaGetErrorString(e)); }
    return ACM_OK;
}

int acm_bubble_diag(acm_ctx* c, double out_host[7])
{
    if (!out_host) return fail(ACM_EINVAL, "acm_bubble_diag: out_host is NULL");
    double sums[DIAG_WIDTH];
    int rc = acm_bubble_sums(c, sums);
    if (rc) return rc;
    out_host[0] = sums[0];
    for (int k = 1; k < DIAG_WIDTH; ++k) out_host[k] = sums[k] / sums[0];
    for (int k = 0; k < DIAG_WIDTH; ++k)
        if (!std::isfinite(out_host[k])) return fail(ACM_EUNSTABLE, "acm_bubble_diag: not finite (no light phase, or diverged)");
    return ACM_OK;
}

int acm_bubble_params(double Re_Gr, double Eo, double D, double t_ref, double rho_H, double rho_star, double mu_star,
                      double out_host[5])
{
    if (!out_host) return fail(ACM_EINVAL, "acm_bubble_params: out_host is NULL");
    if (!(Re_Gr > 0.0) || !(Eo > 0.0) || !(D > 0.0) || !(t_ref > 0.0) || !(rho_H > 0.0) || !(rho_star > 0.0) || !(mu_star > 0.0))
        return fail(ACM_EINVAL, "acm_bubble_params: all arguments must be positive");
    const double g = D / (t_ref * t_ref);                          // eq. 33
    const double mu_H = rho_H * std::sqrt(g * D * D * D) / Re_Gr;   // eq. 31
    const double rho_L = rho_H / rho_star;
    out_host[0] = g;
    out_host[1] = g * rho_H * D * D / Eo;                           // eq. 32
    out_host[2] = mu_H / rho_H;
    out_host[3] = (mu_H / mu_star) / rho_L;
    out_host[4] = rho_L;
    return ACM_OK;
}

double acm_drag_lbm(double g_y, double rho_H, double rho_L, double D, double u_t)
{
    return 4.0 * g_y * (rho_H - rho_L) * D / (3.0 * rho_H * u_t * u_t);
}

double acm_drag_exp(double Re_Gr)
{
    const double a = std::pow(2.67, 0.9), b = std::pow(16.0 / Re_Gr, 0.9);
    return std::pow(a + b, 10.0 / 9.0);
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
    if (c->options & ACM_OPT_MOMENTS)
        return fail(ACM_EINVAL, "acm_set_pdfs: not available with ACM_OPT_MOMENTS (arbitrary populations have no moment representation)");
    int rc = ACM_OK;
    const bool inplace = (c->options & ACM_OPT_INPLACE) != 0;
    if (h) {
        // post-collision convention: two-grid stores it as is (ST_POST); in place as ST_SWAP
        if (inplace) { rc = c->precision == ACM_F64 ? import_h_t<double>(c, h) : import_h_t<float>(c, h); c->stH = ST_SWAP; }
        else if (c->ref == 0.0) rc = copy_async(c, c->ws + c->offH[c->curH], h, (size_t)c->Qh * c->N * c->esz, cudaMemcpyDeviceToDevice, "acm_set_pdfs(h)");
        else rc = check_launch(c, "shift_pop_kernel", launch_shift_pop<float>(c->Qh, aux_launch(c), (const float*)h, wsp<float>(c, c->offH[c->curH]), geom_of(c), c->N, (float)-c->ref));
    }
    if (!rc && g) {
        // incoming convention: in place stores it as is (ST_IN); two-grid pre-shifts it into ST_POST
        if (inplace) { rc = copy_async(c, c->ws + c->offG[c->curG], g, (size_t)c->Qg * c->N * c->esz, cudaMemcpyDeviceToDevice, "acm_set_pdfs(g)"); c->stG = ST_IN; }
        else rc = c->precision == ACM_F64 ? import_g_t<double>(c, g) : import_g_t<float>(c, g);
    }
    return rc;
}

// private stream and events of acm_run_host (created on first use)
static bool io_ready(acm_ctx* c)
{
    if (c->io_stream) return true;
    if (cudaStreamCreateWithFlags(&c->io_stream, cudaStreamNonBlocking) != cudaSuccess) { c->io_stream = nullptr; cudaGetLastError(); return false; }
    for (auto& e : c->io_ev)
        if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return false; }
    return true;
}

// record `ev` on `from` and make `to` wait for it
static int chain(acm_ctx* c, cudaEvent_t ev, cudaStream_t from, cudaStream_t to)
{
    cudaError_t e = cudaEventRecord(ev, from);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(to, ev, 0);
    if (e != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "acm_run_host: %s", cudaGetErrorString(e)); }
    return ACM_OK;
}

int acm_run_host(acm_ctx* c, const void* phi_host, const void* u_host, int n, void* phi_out_host, void* u_out_host,
                 void* p_out_host)
{
    ACM_CHECK_CTX(c);
    if (!phi_host || !u_host) return fail(ACM_EINVAL, "acm_run_host: phi_host and u_host are required");
    if (n < 0) return fail(ACM_EINVAL, "acm_run_host: n must be >= 0");
    if (c->ghost) return fail(ACM_ESTATE, "acm_run_host: not available for a slab (its steps need the halo exchange)");
    const size_t fb = c->N * c->esz;
    char* st = c->ws + c->offStage;
    int rc = copy_async(c, st, phi_host, fb, cudaMemcpyHostToDevice, "acm_run_host(h2d phi)");
    if (!rc) rc = copy_async(c, st + fb, u_host, 3 * fb, cudaMemcpyHostToDevice, "acm_run_host(h2d u)");
    if (!rc) rc = acm_init(c, st, st + fb);
    if (rc) return rc;
    // Results go out on the private stream, each as soon as it is final: phi after the last phase-field kernel (under
    // the last hydrodynamic kernel and the pressure export), u after the last hydrodynamic kernel, p after its export.
    const bool overlap = n > 0 && io_ready(c);
    const cudaStream_t main = c->stream, out = overlap ? c->io_stream : c->stream;
    auto d2h = [&](void* dst, const void* src, size_t bytes, const char* what) {
        cudaError_t e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, out);
        if (e != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "%s: %s", what, cudaGetErrorString(e)); }
        return (int)ACM_OK;
    };
    auto phi_out = [&]() {
        if (!phi_out_host) return (int)ACM_OK;
        const char* src = c->ws + c->offC[c->curC];
        if (c->ref != 0.0) {      // un-shift phi into the staging area first (its phi/u slots are free after acm_init)
            cudaError_t e = launch_shift_field<float>(out, (const float*)src, (float*)st, c->N, (float)c->ref);
            int r = check_launch(c, "acm_run_host(phi)", e);
            if (r) return r;
            src = st;
        }
        return d2h(phi_out_host, src, fb, "acm_run_host(d2h phi)");
    };
    if (overlap) {
        rc = acm_step(c, n - 1);
        if (!rc) rc = c->precision == ACM_F64 ? launch_phase_step<double>(c) : launch_phase_step<float>(c);
        if (!rc) rc = chain(c, c->io_ev[0], main, out);
        if (!rc) rc = phi_out();
        if (!rc) rc = c->precision == ACM_F64 ? launch_hydro_step<double>(c) : launch_hydro_step<float>(c);
        if (!rc && u_out_host) {
            rc = chain(c, c->io_ev[1], main, out);
            if (!rc) rc = d2h(u_out_host, c->ws + c->offU[c->curU], 3 * fb, "acm_run_host(d2h u)");
        }
        if (!rc && p_out_host) {
            rc = acm_fields(c, nullptr, nullptr, st + 4 * fb);
            if (!rc) rc = chain(c, c->io_ev[2], main, out);
            if (!rc) rc = d2h(p_out_host, st + 4 * fb, fb, "acm_run_host(d2h p)");
        }
        if (!rc) rc = chain(c, c->io_ev[3], out, main);      // the context's stream is complete when the copies are
    } else {
        rc = acm_step(c, n);
        if (!rc && p_out_host) rc = acm_fields(c, nullptr, nullptr, st + 4 * fb);
        if (!rc) rc = phi_out();
        if (!rc && u_out_host) rc = d2h(u_out_host, c->ws + c->offU[c->curU], 3 * fb, "acm_run_host(d2h u)");
        if (!rc && p_out_host) rc = d2h(p_out_host, st + 4 * fb, fb, "acm_run_host(d2h p)");
    }
    if (rc) return rc;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { c->sticky = ACM_ECUDA; return fail(ACM_ECUDA, "acm_run_host: %s", cudaGetErrorString(e)); }
    return ACM_OK;
}

}  // extern "C"
