// Host side of the C ABI declared in include/tcp.h: workspace layout, launches, copies.
// There is no CPU path: every entry point that computes launches CUDA kernels.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "../../include/tcp.h"

#include "tcp_halo.cuh"
#include "tcp_launch.h"
#include "tcp_rk.cuh"

namespace {

thread_local char g_err[512];

int fail(int code, const char* fmt, const char* detail = "") {
    std::snprintf(g_err, sizeof g_err, fmt, detail);
    return code;
}
int cuda_fail(cudaError_t e, const char* where) {
    std::snprintf(g_err, sizeof g_err, "%s: %s", where, cudaGetErrorString(e));
    (void)cudaGetLastError();   // reported here: a non-sticky error (a refused cudaMalloc) must not resurface in the next call's launch check
    return e == cudaErrorMemoryAllocation ? TCP_ENOMEM : TCP_ECUDA;
}
#define CK(call)                                                  \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);       \
    } while (0)

constexpr size_t kAlign = 256;
size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

int thermal_q(int thermal) {
    switch (thermal) {
    case TCP_THERMAL_LB_D3Q7: return 7;
    case TCP_THERMAL_LB_D3Q15: return 15;
    case TCP_THERMAL_LB_D3Q19: return 19;
    case TCP_THERMAL_LB_D3Q27: return 27;
    default: return 0;
    }
}

// byte offsets of every array inside the workspace
struct Layout {
    size_t h[2], g[2], f[2], phi[2], T[2], u, rk[3], wallT[3][2], q, total;
};

int validate(int nx, int ny, int nz, const tcp_params* p) {
    if (!p) return fail(TCP_EINVAL, "params is NULL");
    if (p->struct_size != sizeof(tcp_params)) return fail(TCP_EINVAL, "tcp_params.struct_size != sizeof(tcp_params)");
    if (nx < 1 || ny < 1 || nz < 1) return fail(TCP_EINVAL, "extents must be >= 1");
    // cell indices are 32-bit, and so is the offset of a population from the base of its group of 9 planes (tcp_step.cuh): 10 N < 2^32
    if ((double)nx * ny * nz > 429496729.0) return fail(TCP_EINVAL, "nx*ny*nz must be <= 429 496 729 (10 nx ny nz < 2^32)");
    if (ny > 65535 * 8 || nz > 65535) return fail(TCP_EINVAL, "ny must be <= 524280 and nz <= 65535 (grid limits)");
    const int n[3] = {nx, ny, nz};
    for (int a = 0; a < 3; ++a) {
        if (p->bc[a] != TCP_BC_PERIODIC && p->bc[a] != TCP_BC_WALLS) return fail(TCP_EINVAL, "bc must be TCP_BC_PERIODIC or TCP_BC_WALLS");
        if (p->bc[a] == TCP_BC_WALLS && n[a] < 2) return fail(TCP_EINVAL, "a WALLS axis needs at least 2 cells");
    }
    if (p->precision != TCP_F64 && p->precision != TCP_F32) return fail(TCP_EINVAL, "bad precision");
    if (p->thermal < TCP_THERMAL_LB_D3Q7 || p->thermal > TCP_THERMAL_RK4) return fail(TCP_EINVAL, "bad thermal variant");
    if (p->streaming != TCP_STREAM_TWO_GRID && p->streaming != TCP_STREAM_AA) return fail(TCP_EINVAL, "bad streaming pattern");
    if (!(p->tau_H > -0.5) || !(p->tau_L > -0.5)) return fail(TCP_EINVAL, "tau must be > -1/2");
    if (!(p->M > 0) || !(p->xi > 0)) return fail(TCP_EINVAL, "M and xi must be > 0");
    if (!(p->rho_H > 0) || !(p->rho_L > 0)) return fail(TCP_EINVAL, "rho must be > 0");
    if (!(p->kappa_H > 0) || !(p->kappa_L > 0) || !(p->cp_H > 0) || !(p->cp_L > 0)) return fail(TCP_EINVAL, "kappa and cp must be > 0");
    // eps_normal = 0 would make n = grad phi / |grad phi| a 0/0 in every uniform bulk cell (reading S8): a caller who
    // zero-initialises the struct gets an error, not NaNs; tcp_params_default() fills the documented defaults
    if (!(p->eps_normal > 0)) return fail(TCP_EINVAL, "eps_normal must be > 0 (default 1e-32, see tcp_params_default)");
    if (!(p->s_bulk > 0 && p->s_bulk < 2) || !(p->s_high > 0 && p->s_high < 2)) return fail(TCP_EINVAL, "s_bulk and s_high must lie in (0, 2) (default 1, see tcp_params_default)");
    for (int a = 0; a < 3; ++a)
        for (int fc = 0; fc < 2; ++fc)
            if (!(p->wall_contact_angle[a][fc] >= 0.0 && p->wall_contact_angle[a][fc] <= 180.0))
                return fail(TCP_EINVAL, "wall_contact_angle must lie in [0, 180] degrees (default 90, see tcp_params_default)");
    if (p->equilibrium != TCP_EQ_SECOND_ORDER && p->equilibrium != TCP_EQ_MAXWELLIAN) return fail(TCP_EINVAL, "equilibrium must be TCP_EQ_SECOND_ORDER or TCP_EQ_MAXWELLIAN");
    if (p->equilibrium == TCP_EQ_MAXWELLIAN) {
        const int qt = thermal_q(p->thermal);
        if (p->hydro_lattice != 27 || (qt != 0 && qt != 27))
            return fail(TCP_EUNSUPPORTED, "Maxwellian equilibrium: D3Q27 lattices only (hydro_lattice = 27; thermal D3Q27 LB, RK2 or RK4)");
        if (p->high_rate_equals_shear || p->s_high != 1.0)
            return fail(TCP_EUNSUPPORTED, "Maxwellian equilibrium: with the closed-form collision only (s_high = 1, high_rate_equals_shear = 0)");
    }
    if (p->collision_space != TCP_SPACE_CENTRAL && p->collision_space != TCP_SPACE_RAW) return fail(TCP_EINVAL, "collision_space must be TCP_SPACE_CENTRAL or TCP_SPACE_RAW");
    if (p->hydro_lattice != 27 && p->hydro_lattice != 19) return fail(TCP_EINVAL, "hydro_lattice must be 27 or 19 (default 27, see tcp_params_default)");
    if (p->hydro_lattice == 19 && p->s_high != 1.0 && !p->high_rate_equals_shear)
        return fail(TCP_EUNSUPPORTED, "hydro_lattice = 19: the closed-form central-moment collision (s_high = 1) and BGK only; general rates need the D3Q27 basis");
    if (p->high_rate_equals_shear != 0 && p->high_rate_equals_shear != 1) return fail(TCP_EINVAL, "high_rate_equals_shear must be 0 or 1");
    return TCP_OK;
}

Layout make_layout(int nx, int ny, int nz, const tcp_params* p) {
    Layout L;
    std::memset(&L, 0, sizeof L);
    const size_t es = p->precision == TCP_F64 ? 8 : 4;
    const size_t N = (size_t)nx * ny * nz;
    const int QT = thermal_q(p->thermal);
    size_t off = 0;
    auto take = [&](size_t count) { size_t o = off; off = align_up(off + count * es); return o; };
    const bool aa = p->streaming == TCP_STREAM_AA;      // in-place streaming: one grid of populations
    for (int b = 0; b < 2; ++b) L.h[b] = (aa && b) ? L.h[0] : take(27 * N);
    for (int b = 0; b < 2; ++b) L.g[b] = (aa && b) ? L.g[0] : take((size_t)p->hydro_lattice * N);
    for (int b = 0; b < 2; ++b) L.f[b] = QT ? ((aa && b) ? L.f[0] : take((size_t)QT * N)) : 0;
    for (int b = 0; b < 2; ++b) L.phi[b] = take(N);
    for (int b = 0; b < 2; ++b) L.T[b] = take(N);
    L.u = take(3 * N);
    const int nrk = p->thermal == TCP_THERMAL_RK2 ? 1 : (p->thermal == TCP_THERMAL_RK4 ? 3 : 0);
    for (int k = 0; k < nrk; ++k) L.rk[k] = take(N);
    const size_t plane[3] = {(size_t)ny * nz, (size_t)nx * nz, (size_t)nx * ny};
    for (int a = 0; a < 3; ++a)
        for (int fc = 0; fc < 2; ++fc) L.wallT[a][fc] = take(plane[a]);
    L.q = take(N);
    L.total = off;
    return L;
}

}  // namespace

struct tcp_sim {
    int nx, ny, nz;
    size_t N;
    tcp_params P;
    Layout L;
    char* base;
    bool owns_memory, owns_stream;
    cudaStream_t stream;
    int cur;                 // index of the h, g, phi buffers holding time level n
    int curT;                // same for f and T (they advance alone in tcp_relax_temperature)
    bool initialised, has_q, walls, stepped;
    long long launches;
    cudaEvent_t ev0, ev1;
    cudaEvent_t evc0, evc1;  // tcp_pattern_copy_ms only: the calibration must not disturb tcp_last_step_ms
    int device;              // the CUDA device the workspace lives on; every entry point runs with it current
    bool use_pair;           // fp32: two cells per thread, packed arithmetic (x periodic, nx even)
    int aa_next;             // AA streaming: type of the next step (1 even, 2 odd); 0 = two-grid
    // z-slab of a decomposed box (tcp_set_halo): plane 0 / nz-1 is a ghost plane filled from a neighbour
    bool halo[2];
    bool in_step;            // between tcp_step_begin and the tcp_step_advance / tcp_step_end that completes the step
    int phase;               // whose message is in flight (0 fused kernel, k = Runge-Kutta stage k)
    cudaStream_t comm;       // caller's stream for pack / exchange / unpack
    void* send[2];           // caller's device buffers, one message each
    void* recv[2];
    cudaEvent_t ev_bnd, ev_comm;
};

// ---- tcp_read_pressure_static: scratch that no call allocates -------------------------------------------------------
// File-scope device array (8 MiB on every GPU that loads the library, until exit).  In HOST code `g_static_scratch` is
// only a stand-in for the symbol, not a device address: the address is resolved once per device, with that device
// current, by cudaGetSymbolAddress in tcp_read_pressure_static, and that pointer is what the kernel gets.
static __device__ __align__(256) unsigned char g_static_scratch[TCP_STATIC_SCRATCH_BYTES];
static void* g_static_scratch_addr[tcp::kMaxDevices] = {};

namespace {

template <typename real> real* ptr(const tcp_sim* s, size_t off) { return reinterpret_cast<real*>(s->base + off); }

// Makes the simulation's device current for the duration of an entry point and restores the caller's afterwards,
// so that several simulations on several GPUs can be driven from one thread.
struct DeviceScope {
    int prev = -1;
    bool switched = false;
    explicit DeviceScope(const tcp_sim* s) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != s->device) switched = cudaSetDevice(s->device) == cudaSuccess;
    }
    ~DeviceScope() { if (switched) cudaSetDevice(prev); }
};

// constants {m, s1, s2} of tcp::fast_div for the divisor d >= 1
void fast_div_make(unsigned d, unsigned c[3]) {
    unsigned l = 0;
    while ((1ull << l) < d) ++l;                       // l = ceil(log2 d)
    c[0] = (unsigned)(((1ull << 32) * ((1ull << l) - d)) / d + 1);
    c[1] = l < 1 ? l : 1;
    c[2] = l > 1 ? l - 1 : 0;
}

template <typename real>
tcp::StepArgs<real> make_args(const tcp_sim* s) {
    tcp::StepArgs<real> A;
    std::memset(&A, 0, sizeof A);
    const tcp_params& P = s->P;
    const int c = s->cur, o = 1 - s->cur, cT = s->curT, oT = 1 - s->curT;
    A.nx = s->nx; A.ny = s->ny; A.nz = s->nz; A.ncell = (int)s->N;
    A.cell0 = 0; A.cell1 = (int)s->N;
    A.aa = s->aa_next;
    for (int a = 0; a < 3; ++a) A.wall[a] = P.bc[a] == TCP_BC_WALLS;
    A.h_in = ptr<real>(s, s->L.h[c]); A.h_out = ptr<real>(s, s->L.h[o]);
    A.g_in = ptr<real>(s, s->L.g[c]); A.g_out = ptr<real>(s, s->L.g[o]);
    A.f_in = ptr<real>(s, s->L.f[cT]); A.f_out = ptr<real>(s, s->L.f[oT]);
    A.phi_in = ptr<real>(s, s->L.phi[c]); A.phi_out = ptr<real>(s, s->L.phi[o]);
    A.T_in = ptr<real>(s, s->L.T[cT]); A.T_out = ptr<real>(s, s->L.T[oT]);
    A.u = ptr<real>(s, s->L.u);
    A.q_src = s->has_q ? ptr<real>(s, s->L.q) : nullptr;
    for (int a = 0; a < 3; ++a)
        for (int fc = 0; fc < 2; ++fc) A.wallT[a][fc] = ptr<real>(s, s->L.wallT[a][fc]);
    A.rho_L = (real)P.rho_L; A.drho = (real)(P.rho_H - P.rho_L);
    A.tau_L = (real)P.tau_L; A.dtau = (real)(P.tau_H - P.tau_L);
    A.xi = (real)P.xi; A.w_phi = (real)(1.0 / (0.5 + 3.0 * P.M));
    A.inv_xi = (real)(1.0 / P.xi);
    fast_div_make((unsigned)s->nx, A.div_nx);
    fast_div_make((unsigned)s->ny, A.div_ny);
    fast_div_make((unsigned)(s->nx > 1 ? s->nx / 2 : 1), A.div_hx);
    A.sigma_ref = (real)P.sigma_ref; A.sigma_T = (real)P.sigma_T; A.T_ref = (real)P.T_ref; A.sigma_TT = (real)P.sigma_TT;
    A.kappa_L = (real)P.kappa_L; A.dkappa = (real)(P.kappa_H - P.kappa_L);
    A.cp_L = (real)P.cp_L; A.dcp = (real)(P.cp_H - P.cp_L);
    for (int a = 0; a < 3; ++a) A.grav[a] = (real)P.gravity[a];
    A.s_bulk = (real)P.s_bulk;
    A.s_high = (real)P.s_high;
    A.moving = 0;
    for (int a = 0; a < 3; ++a)
        for (int fc = 0; fc < 2; ++fc)
            for (int k = 0; k < 3; ++k) {
                A.wall_u[a][fc][k] = (real)P.wall_u[a][fc][k];
                if (P.wall_u[a][fc][k] != 0.0) A.moving = 1;
            }
    A.cm_frame = (real)(P.collision_space == TCP_SPACE_RAW ? 0.0 : 1.0);
    A.maxwell = P.equilibrium == TCP_EQ_MAXWELLIAN;
    A.eq_sigma = (real)(A.maxwell ? 0.0 : 1.0);
    // wetting (reading S20): a = -(2 / xi) cos(theta) per wall; exactly 0 for the neutral 90 degrees
    A.wetting = 0;
    for (int a = 0; a < 3; ++a)
        for (int fc = 0; fc < 2; ++fc) {
            const double th = P.wall_contact_angle[a][fc];
            const double wa = (th == 90.0 || P.bc[a] != TCP_BC_WALLS) ? 0.0 : -(2.0 / P.xi) * std::cos(th * 3.14159265358979323846 / 180.0);
            A.wet_a[a][fc] = (real)wa;
            if (wa != 0.0) A.wetting = 1;
        }
    // S8: eps keeps n = grad phi / |grad phi| finite where grad phi vanishes.  In fp32 a gradient
    // below ~1e-6 is round-off of phi ~ 1, and a round-off-directed sharpening flux makes phi = 0 / 1
    // unstable to noise (measured: 1e-4 error after 100 steps next to a wall), so eps is floored there.
    A.eps = (real)(sizeof(real) == 4 ? std::fmax(P.eps_normal, 1e-12) : P.eps_normal);
    return A;
}

unsigned grid_for(size_t n) { return (unsigned)((n + tcp::kBlock - 1) / tcp::kBlock); }

// the z-marching stage kernel is instantiated per (walls, RkArgs::mode, heat source present, kappa_H != kappa_L)
template <typename real, bool WALLS, int MODE, bool HAS_Q, bool HAS_DK>
void launch_rk_march_inst(const tcp_sim* s, const tcp::RkArgs<real>& R, dim3 grid, dim3 block) {
    auto kern = tcp::rk_stage_march_kernel<real, WALLS, MODE, HAS_Q, HAS_DK>;
    const size_t ring_bytes = tcp::rk_ring_bytes<real>();        // cell-data ring (dynamic shared memory)
    static bool configured[tcp::kMaxDevices] = {};               // once per instantiation and device: static + dynamic can exceed 48 KB
    if (!configured[s->device])
        configured[s->device] = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ring_bytes) == cudaSuccess;
    kern<<<grid, block, ring_bytes, s->stream>>>(R);       // a failed attribute call surfaces here as a launch error (cudaGetLastError)
}
template <typename real, bool WALLS, int MODE>
void launch_rk_march_q(const tcp_sim* s, const tcp::RkArgs<real>& R, dim3 grid, dim3 block) {
    const bool dk = s->P.kappa_H != s->P.kappa_L;       // grad kappa . grad T present
    if (R.S.q_src) {
        if (dk) launch_rk_march_inst<real, WALLS, MODE, true, true>(s, R, grid, block);
        else launch_rk_march_inst<real, WALLS, MODE, true, false>(s, R, grid, block);
    } else {
        if (dk) launch_rk_march_inst<real, WALLS, MODE, false, true>(s, R, grid, block);
        else launch_rk_march_inst<real, WALLS, MODE, false, false>(s, R, grid, block);
    }
}
template <typename real, bool WALLS>
void launch_rk_march_w(const tcp_sim* s, const tcp::RkArgs<real>& R, dim3 grid, dim3 block) {
    switch (R.mode) {
    case 0: launch_rk_march_q<real, WALLS, 0>(s, R, grid, block); break;
    case 1: launch_rk_march_q<real, WALLS, 1>(s, R, grid, block); break;
    case 2: launch_rk_march_q<real, WALLS, 2>(s, R, grid, block); break;
    default: launch_rk_march_q<real, WALLS, 3>(s, R, grid, block); break;
    }
}
template <typename real>
void launch_rk_march(const tcp_sim* s, const tcp::RkArgs<real>& R, dim3 grid, dim3 block) {
    if (s->walls) launch_rk_march_w<real, true>(s, R, grid, block);
    else launch_rk_march_w<real, false>(s, R, grid, block);
}

template <typename real>
void launch_rk_stage(const tcp_sim* s, const tcp::RkArgs<real>& R) {
    const int P = s->nx * s->ny, planes = (R.S.cell1 - R.S.cell0) / P;       // whole planes [cell0, cell1)
    const dim3 block(tcp::kRkTX, tcp::kRkTY);                                 // z-marching tile kernel (tcp_rk.cuh)
    const dim3 grid((s->nx + tcp::kRkTX - 1) / tcp::kRkTX, (s->ny + tcp::kRkTY - 1) / tcp::kRkTY, (planes + tcp::kRkCZ - 1) / tcp::kRkCZ);
    launch_rk_march<real>(s, R, grid, block);
}

// The stages of the Runge-Kutta update of T (eqs. 25-26) from T[curT] into T[1 - curT], in order;
// phi = the phi to differentiate.  Returns their number (0 on the thermal LB paths).
template <typename real>
int rk_stages(const tcp_sim* s, const tcp::StepArgs<real>& A, const real* phi, tcp::RkArgs<real> st[4]) {
    const int th = s->P.thermal;
    if (th != TCP_THERMAL_RK2 && th != TCP_THERMAL_RK4) return 0;
    tcp::RkArgs<real> R;
    std::memset(&R, 0, sizeof R);
    R.S = A;
    R.S.phi_in = phi;
    real* Tn = ptr<real>(s, s->L.T[s->curT]);
    real* Tnew = ptr<real>(s, s->L.T[1 - s->curT]);
    real* Ya = ptr<real>(s, s->L.rk[0]);
    R.Tn = Tn;
    if (th == TCP_THERMAL_RK2) {         // eq. 26 (G6)
        R.Y = Tn; R.out = Ya; R.c_out = (real)0.5; R.mode = 0;
        st[0] = R;
        R.Y = Ya; R.out = Tnew; R.c_out = (real)1.0; R.mode = 0;
        st[1] = R;
        return 2;
    }
    real* Yb = ptr<real>(s, s->L.rk[1]);   // eq. 25
    real* acc = ptr<real>(s, s->L.rk[2]);
    R.acc_in = acc; R.acc_out = acc;
    R.Y = Tn; R.out = Ya; R.c_out = (real)0.5; R.c_acc = (real)(1.0 / 6.0); R.mode = 1;
    st[0] = R;
    R.Y = Ya; R.out = Yb; R.c_out = (real)0.5; R.c_acc = (real)(1.0 / 3.0); R.mode = 2;
    st[1] = R;
    R.Y = Yb; R.out = Ya; R.c_out = (real)1.0; R.c_acc = (real)(1.0 / 3.0); R.mode = 2;
    st[2] = R;
    R.Y = Ya; R.out = Tnew; R.c_acc = (real)(1.0 / 6.0); R.mode = 3;
    st[3] = R;
    return 4;
}

// Stage 1 inside the fused kernel (rk_stage1_local, tcp_step.cuh): the Runge-Kutta paths with equal conductivities.
bool rk_first_stage_fused(const tcp_sim* s) {
    const int th = s->P.thermal;
    if (th != TCP_THERMAL_RK2 && th != TCP_THERMAL_RK4) return false;
    return s->P.kappa_H == s->P.kappa_L;
}

// stages [first, n) of the Runge-Kutta update
template <typename real>
void rk_update(tcp_sim* s, const tcp::StepArgs<real>& A, const real* phi, int first = 0) {
    tcp::RkArgs<real> st[4];
    const int n = rk_stages<real>(s, A, phi, st);
    for (int i = first; i < n; ++i) launch_rk_stage<real>(s, st[i]);
    s->launches += n > first ? n - first : 0;
}

// hand the fused kernel the outputs of stage 1 (Y1, and the RK4 accumulator)
template <typename real>
void attach_first_stage(tcp_sim* s, tcp::StepArgs<real>& A) {
    tcp::RkArgs<real> st[4];
    if (rk_stages<real>(s, A, A.phi_out, st) == 0) return;
    A.rk1_out = st[0].out; A.rk1_c_out = st[0].c_out;
    A.rk1_acc = st[0].mode == 1 ? st[0].acc_out : nullptr; A.rk1_c_acc = st[0].c_acc;
}

// temperature update alone, phi / u / h~ / g~ frozen
template <typename real>
int relax_t(tcp_sim* s, int nsteps) {
    const int qt = thermal_q(s->P.thermal);
    int aa = s->aa_next;                       // parity of the thermal populations during the relaxation
    for (int n = 0; n < nsteps; ++n) {
        tcp::StepArgs<real> A = make_args<real>(s);
        if (qt) {
            tcp::FusedCfg c;
            c.qt = qt; c.walls = s->walls; c.mode = s->P.equilibrium == TCP_EQ_MAXWELLIAN ? 4 : (s->P.high_rate_equals_shear ? 1 : 0); c.aa = aa; c.device = s->device; c.grid = grid_for(s->N);
            CK(s->walls ? tcp::launch_thermal_walls(c, A, s->stream) : tcp::launch_thermal_periodic(c, A, s->stream));
            s->launches++;
            if (aa) aa = 3 - aa;
        } else {
            rk_update<real>(s, A, A.phi_in);
        }
        s->curT = 1 - s->curT;
    }
    CK(cudaGetLastError());
    return TCP_OK;
}

// the fused phase + hydro (+ thermal LB) kernel on the cells [A.cell0, A.cell1)
template <typename real>
int launch_fused(tcp_sim* s, const tcp::StepArgs<real>& A) {
    // collision mode: 0 closed-form central moments (s_high = 1), 1 BGK, 2 general rates (full transform)
    const int mode = s->P.equilibrium == TCP_EQ_MAXWELLIAN ? 4 : (s->P.high_rate_equals_shear ? 1 : (s->P.s_high != 1.0 ? 2 : 0));
    tcp::FusedCfg c;
    c.qt = thermal_q(s->P.thermal); c.walls = s->walls; c.mode = mode; c.aa = s->aa_next; c.device = s->device;
    c.grid = grid_for((size_t)(A.cell1 - A.cell0));
    const bool q19 = s->P.hydro_lattice == 19;       // D3Q19 hydrodynamic lattice: kernels of the *_q19 translation units
    if constexpr (sizeof(real) == 4) {
        if (s->use_pair && (mode == 0 || mode == 4)) {
            if (q19) CK(s->walls ? tcp::launch_pair_walls_q19(c, A, s->stream) : tcp::launch_pair_periodic_q19(c, A, s->stream));
            else CK(s->walls ? tcp::launch_pair_walls(c, A, s->stream) : tcp::launch_pair_periodic(c, A, s->stream));
            s->launches++;
            return TCP_OK;
        }
    }
    if (q19) CK(s->walls ? tcp::launch_fused_walls_q19(c, A, s->stream) : tcp::launch_fused_periodic_q19(c, A, s->stream));
    else CK(s->walls ? tcp::launch_fused_walls(c, A, s->stream) : tcp::launch_fused_periodic(c, A, s->stream));
    s->launches++;
    return TCP_OK;
}

// one time step: Algorithm 1 (thermal LB, one fused kernel) or Algorithm 2 (fused phase+hydro
// kernel, then the Runge-Kutta stages)
template <typename real>
int step_once(tcp_sim* s) {
    tcp::StepArgs<real> A = make_args<real>(s);
    const bool fused1 = rk_first_stage_fused(s);
    if (fused1) attach_first_stage<real>(s, A);
    int rc = launch_fused<real>(s, A);
    if (rc) return rc;
    A.rk1_out = nullptr; A.rk1_acc = nullptr;
    rk_update<real>(s, A, A.phi_out, fused1 ? 1 : 0);        // phi^{n+1}; u already holds u^{n+1}
    s->cur = 1 - s->cur;
    s->curT = 1 - s->curT;
    if (s->aa_next) s->aa_next = 3 - s->aa_next;
    return TCP_OK;
}

// ---- z-slab with ghost planes (tcp_set_halo): Algorithm 1 / 2's order -- boundary cells first, their
// values on the way to the neighbour while the interior is updated.  A step has one
// phase on the thermal LB paths (the fused kernel) and 1 + the number of stages on the Runge-Kutta paths
// (fused phase + hydro kernel, then every stage: its output is differentiated by the next one) ------------

int halo_phases(const tcp_sim* s) {
    const int stages = s->P.thermal == TCP_THERMAL_RK2 ? 2 : (s->P.thermal == TCP_THERMAL_RK4 ? 4 : 0);
    return 1 + stages - (rk_first_stage_fused(s) ? 1 : 0);
}

// The arrays (pointers to their plane z = 0) of which one z-plane travels in direction dir (+1 up, -1 down)
// after phase p: [h~ c_z=dir][g~ c_z=dir][f~ c_z=dir][phi][T] of the new time level, or the stage's output.
template <typename real>
int phase_message(const tcp_sim* s, int p, int dir, real* fields[32]) {
    const size_t N = s->N;
    const int o = 1 - s->cur, oT = 1 - s->curT;
    int m = 0;
    const int f1 = rk_first_stage_fused(s) ? 1 : 0;
    if (p > 0) {
        tcp::RkArgs<real> st[4];
        rk_stages<real>(s, make_args<real>(s), nullptr, st);
        fields[m++] = st[p - 1 + f1].out;
        return m;
    }
    for (int q = 0; q < 27; ++q)
        if (tcp::cz27(q) == dir) fields[m++] = ptr<real>(s, s->L.h[o]) + q * N;
    const int QH = s->P.hydro_lattice;
    for (int k = 0; k < QH; ++k)
        if (tcp::cz27(tcp::q_of(QH, k)) == dir) fields[m++] = ptr<real>(s, s->L.g[o]) + k * N;
    const int QT = thermal_q(s->P.thermal);
    for (int k = 0; k < QT; ++k)
        if (tcp::cz27(tcp::q_of(QT, k)) == dir) fields[m++] = ptr<real>(s, s->L.f[oT]) + k * N;
    fields[m++] = ptr<real>(s, s->L.phi[o]);
    if (QT) fields[m++] = ptr<real>(s, s->L.T[oT]);
    if (f1) {   // stage 1 ran inside the fused kernel: its output travels with this message
        tcp::RkArgs<real> st[4];
        rk_stages<real>(s, make_args<real>(s), nullptr, st);
        fields[m++] = st[0].out;
    }
    return m;
}

// `gather`: plane z of the travelling arrays -> message; otherwise message -> plane z
template <typename real>
void halo_planes(const tcp_sim* s, tcp::HaloCopy& C, int p, int dir, int z, void* message, bool gather) {
    const size_t P = (size_t)s->nx * s->ny;
    real* fields[32];
    const int m = phase_message<real>(s, p, dir, fields);
    for (int i = 0; i < m; ++i) {
        real* plane = fields[i] + (size_t)z * P;
        real* in_msg = static_cast<real*>(message) + (size_t)i * P;
        C.src[C.nplanes] = gather ? plane : in_msg;
        C.dst[C.nplanes] = gather ? in_msg : plane;
        C.nplanes++;
    }
}

template <typename real>
int halo_copy(tcp_sim* s, const tcp::HaloCopy& C) {
    if (C.nplanes == 0) return TCP_OK;
    const dim3 grid((unsigned)((C.plane_cells + 255) / 256), (unsigned)C.nplanes);
    tcp::halo_copy_kernel<real><<<grid, 256, 0, s->comm>>>(C);
    s->launches++;
    CK(cudaGetLastError());
    return TCP_OK;
}

// phase p: its kernel on the boundary planes, the gather of their new values (comm stream), its kernel on the interior
template <typename real>
int phase_begin(tcp_sim* s, int p) {
    const int P = s->nx * s->ny;
    const int zlo = s->halo[0] ? 1 : 0, zhi = s->nz - 1 - (s->halo[1] ? 1 : 0);   // first / last plane this slab owns
    tcp::StepArgs<real> A = make_args<real>(s);
    auto planes = [&](int z0, int z1) {       // run the phase on the planes z0..z1
        if (z1 < z0) return (int)TCP_OK;
        A.cell0 = z0 * P; A.cell1 = (z1 + 1) * P;
        const int f1 = rk_first_stage_fused(s) ? 1 : 0;
        if (p == 0) {
            if (f1) attach_first_stage<real>(s, A);
            const int r = launch_fused<real>(s, A);
            A.rk1_out = nullptr; A.rk1_acc = nullptr;
            return r;
        }
        tcp::RkArgs<real> st[4];
        rk_stages<real>(s, A, A.phi_out, st);
        launch_rk_stage<real>(s, st[p - 1 + f1]);
        s->launches++;
        return (int)TCP_OK;
    };
    int rc = TCP_OK;
    if (s->halo[0]) rc = planes(zlo, zlo);
    if (!rc && s->halo[1] && !(s->halo[0] && zhi == zlo)) rc = planes(zhi, zhi);
    if (rc) return rc;
    CK(cudaEventRecord(s->ev_bnd, s->stream));
    CK(cudaStreamWaitEvent(s->comm, s->ev_bnd, 0));
    tcp::HaloCopy C;
    std::memset(&C, 0, sizeof C);
    C.plane_cells = P;
    if (s->halo[0]) halo_planes<real>(s, C, p, -1, zlo, s->send[0], true);
    if (s->halo[1]) halo_planes<real>(s, C, p, +1, zhi, s->send[1], true);
    rc = halo_copy<real>(s, C);
    if (rc) return rc;
    rc = planes(zlo + (s->halo[0] ? 1 : 0), zhi - (s->halo[1] ? 1 : 0));
    if (rc) return rc;
    CK(cudaGetLastError());
    return TCP_OK;
}

// the message of phase p has been transferred (enqueued on the comm stream): scatter it into the ghost planes
template <typename real>
int phase_end(tcp_sim* s, int p) {
    tcp::HaloCopy C;
    std::memset(&C, 0, sizeof C);
    C.plane_cells = s->nx * s->ny;
    if (s->halo[0]) halo_planes<real>(s, C, p, +1, 0, s->recv[0], false);          // from below, moving up
    if (s->halo[1]) halo_planes<real>(s, C, p, -1, s->nz - 1, s->recv[1], false);  // from above, moving down
    int rc = halo_copy<real>(s, C);
    if (rc) return rc;
    CK(cudaEventRecord(s->ev_comm, s->comm));
    CK(cudaStreamWaitEvent(s->stream, s->ev_comm, 0));
    return TCP_OK;
}

template <typename real>
int step_begin_t(tcp_sim* s) {
    CK(cudaEventRecord(s->ev0, s->stream));
    int rc = phase_begin<real>(s, 0);
    if (rc) return rc;
    s->in_step = true;
    s->phase = 0;
    return TCP_OK;
}

template <typename real>
int step_advance_t(tcp_sim* s, int* transfers_left) {
    int rc = phase_end<real>(s, s->phase);
    if (rc) return rc;
    if (s->phase + 1 < halo_phases(s)) {
        rc = phase_begin<real>(s, s->phase + 1);
        if (rc) return rc;
        s->phase++;
        *transfers_left = halo_phases(s) - s->phase;
        return TCP_OK;
    }
    CK(cudaEventRecord(s->ev1, s->stream));
    s->cur = 1 - s->cur;
    s->curT = 1 - s->curT;
    s->in_step = false;
    s->stepped = true;
    *transfers_left = 0;
    return TCP_OK;
}

template <typename real>
int init_fields_t(tcp_sim* s, const void* phi, const void* u, const void* T) {
    const size_t N = s->N, es = sizeof(real);
    s->cur = 0;
    s->curT = 0;
    CK(cudaMemcpyAsync(ptr<real>(s, s->L.phi[0]), phi, N * es, cudaMemcpyDefault, s->stream));
    if (u) CK(cudaMemcpyAsync(ptr<real>(s, s->L.u), u, 3 * N * es, cudaMemcpyDefault, s->stream));
    else CK(cudaMemsetAsync(ptr<real>(s, s->L.u), 0, 3 * N * es, s->stream));
    if (T) CK(cudaMemcpyAsync(ptr<real>(s, s->L.T[0]), T, N * es, cudaMemcpyDefault, s->stream));
    else {
        tcp::fill_kernel<real><<<(unsigned)((N + 255) / 256), 256, 0, s->stream>>>(ptr<real>(s, s->L.T[0]), (long long)N, (real)s->P.T_ref);
        s->launches++;
    }
    s->aa_next = s->P.streaming == TCP_STREAM_AA ? 1 : 0;   // AA: init stores pushed populations, the first step is an even one
    tcp::StepArgs<real> A = make_args<real>(s);
    A.h_out = ptr<real>(s, s->L.h[0]); A.g_out = ptr<real>(s, s->L.g[0]); A.f_out = ptr<real>(s, s->L.f[0]);
    const unsigned grid = grid_for(N);
    if (s->P.hydro_lattice == 19) {
        switch (thermal_q(s->P.thermal)) {
        case 7: tcp::init_kernel<real, 7, 19><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        case 15: tcp::init_kernel<real, 15, 19><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        case 19: tcp::init_kernel<real, 19, 19><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        case 27: tcp::init_kernel<real, 27, 19><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        default: tcp::init_kernel<real, 0, 19><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        }
    } else {
        switch (thermal_q(s->P.thermal)) {
        case 7: tcp::init_kernel<real, 7><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        case 15: tcp::init_kernel<real, 15><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        case 19: tcp::init_kernel<real, 19><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        case 27: tcp::init_kernel<real, 27><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        default: tcp::init_kernel<real, 0><<<grid, tcp::kBlock, 0, s->stream>>>(A); break;
        }
    }
    s->launches++;
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(s->stream));   // the caller may free its arrays when we return
    s->initialised = true;
    return TCP_OK;
}

template <typename real>
int fill_wall(tcp_sim* s, int axis, int face, const void* Tw) {
    const size_t plane[3] = {(size_t)s->ny * s->nz, (size_t)s->nx * s->nz, (size_t)s->nx * s->ny};
    real* dst = ptr<real>(s, s->L.wallT[axis][face]);
    const int qt = thermal_q(s->P.thermal);
    // AA streaming with the populations in the pushed layout (after tcp_init_fields or an odd step): the wall links of
    // f~ already carry the old plane, see aa_wall_repush_kernel.  The new plane is staged in the spare phi buffer.
    const bool repush = s->P.streaming == TCP_STREAM_AA && s->initialised && s->aa_next == 1 && qt > 0 && s->P.bc[axis] == TCP_BC_WALLS;
    real* target = repush ? ptr<real>(s, s->L.phi[1 - s->cur]) : dst;
    if (Tw) CK(cudaMemcpyAsync(target, Tw, plane[axis] * sizeof(real), cudaMemcpyDefault, s->stream));
    else {
        tcp::fill_kernel<real><<<(unsigned)((plane[axis] + 255) / 256), 256, 0, s->stream>>>(target, (long long)plane[axis],
                                                                                        (real)s->P.wall_T[axis][face]);
        s->launches++;
        CK(cudaGetLastError());
    }
    if (repush) {
        const tcp::StepArgs<real> A = make_args<real>(s);
        real* f = ptr<real>(s, s->L.f[0]);
        const unsigned grid = grid_for(plane[axis]);
        const int pc = (int)plane[axis];
        switch (qt) {
        case 7: tcp::aa_wall_repush_kernel<real, 7><<<grid, tcp::kBlock, 0, s->stream>>>(A, f, axis, face, target, dst, pc); break;
        case 15: tcp::aa_wall_repush_kernel<real, 15><<<grid, tcp::kBlock, 0, s->stream>>>(A, f, axis, face, target, dst, pc); break;
        case 19: tcp::aa_wall_repush_kernel<real, 19><<<grid, tcp::kBlock, 0, s->stream>>>(A, f, axis, face, target, dst, pc); break;
        default: tcp::aa_wall_repush_kernel<real, 27><<<grid, tcp::kBlock, 0, s->stream>>>(A, f, axis, face, target, dst, pc); break;
        }
        s->launches++;
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(dst, target, plane[axis] * sizeof(real), cudaMemcpyDeviceToDevice, s->stream));
    }
    CK(cudaStreamSynchronize(s->stream));
    return TCP_OK;
}

// p = c_s^2 rho(phi) sum_i g~_i into `out` (device memory, N values): natural layout, or the pushed layout of AA streaming
template <typename real>
void launch_pressure(tcp_sim* s, real* out) {
    const size_t N = s->N;
    const real* phi = ptr<real>(s, s->L.phi[s->cur]);
    const real rho_L = (real)s->P.rho_L, drho = (real)(s->P.rho_H - s->P.rho_L);
    const bool q19 = s->P.hydro_lattice == 19;
    if (s->aa_next == 1) {   // AA, populations in the pushed layout (after init or an odd step)
        if (q19) tcp::pressure_pushed_kernel<real, 19><<<grid_for(N), tcp::kBlock, 0, s->stream>>>(make_args<real>(s), ptr<real>(s, s->L.g[0]), phi, out);
        else tcp::pressure_pushed_kernel<real, 27><<<grid_for(N), tcp::kBlock, 0, s->stream>>>(make_args<real>(s), ptr<real>(s, s->L.g[0]), phi, out);
    } else {
        if (q19) tcp::pressure_kernel<real, 19><<<grid_for(N), tcp::kBlock, 0, s->stream>>>(ptr<real>(s, s->L.g[s->cur]), phi, out, (int)N, rho_L, drho);
        else tcp::pressure_kernel<real, 27><<<grid_for(N), tcp::kBlock, 0, s->stream>>>(ptr<real>(s, s->L.g[s->cur]), phi, out, (int)N, rho_L, drho);
    }
    s->launches++;
}

template <typename real>
int read_fields_t(tcp_sim* s, void* phi, void* u, void* p, void* T) {
    const size_t N = s->N, es = sizeof(real);
    if (phi) CK(cudaMemcpyAsync(phi, ptr<real>(s, s->L.phi[s->cur]), N * es, cudaMemcpyDefault, s->stream));
    if (u) CK(cudaMemcpyAsync(u, ptr<real>(s, s->L.u), 3 * N * es, cudaMemcpyDefault, s->stream));
    if (T) CK(cudaMemcpyAsync(T, ptr<real>(s, s->L.T[s->curT]), N * es, cudaMemcpyDefault, s->stream));
    if (p) {
        real* scratch = ptr<real>(s, s->L.phi[1 - s->cur]);   // free between steps
        launch_pressure<real>(s, scratch);
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(p, scratch, N * es, cudaMemcpyDefault, s->stream));
    }
    CK(cudaStreamSynchronize(s->stream));
    return TCP_OK;
}

int create_common(int nx, int ny, int nz, const tcp_params* p, void* workspace, size_t bytes, void* stream, bool own, tcp_sim** out) {
    if (!out) return fail(TCP_EINVAL, "out is NULL");
    *out = nullptr;
    int rc = validate(nx, ny, nz, p);
    if (rc) return rc;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(TCP_ECUDA, "no CUDA device: this library has no CPU path");
    }
    tcp_sim* s = new (std::nothrow) tcp_sim();
    if (!s) return fail(TCP_ENOMEM, "host allocation failed");
    s->nx = nx; s->ny = ny; s->nz = nz; s->N = (size_t)nx * ny * nz; s->P = *p;
    s->L = make_layout(nx, ny, nz, p);
    s->walls = p->bc[0] == TCP_BC_WALLS || p->bc[1] == TCP_BC_WALLS || p->bc[2] == TCP_BC_WALLS;
    s->owns_memory = own; s->owns_stream = own;
    if (own) {
        e = cudaGetDevice(&s->device);
        if (e != cudaSuccess) { delete s; return cuda_fail(e, "cudaGetDevice"); }
    } else {
        // the workspace decides the device: memory and stream of any GPU of the process may be handed in
        if (!workspace) { delete s; return fail(TCP_EINVAL, "workspace is NULL"); }
        cudaPointerAttributes at;
        e = cudaPointerGetAttributes(&at, workspace);
        if (e != cudaSuccess || at.type != cudaMemoryTypeDevice) { cudaGetLastError(); delete s; return fail(TCP_EINVAL, "workspace is not device memory"); }
        s->device = at.device;
    }
    if (s->device < 0 || s->device >= tcp::kMaxDevices) { delete s; return fail(TCP_EUNSUPPORTED, "device ordinal out of range"); }
    DeviceScope scope(s);
    // fp32: the packed-pair kernel wherever its layout rules hold (x periodic, nx even), else one cell per thread
    s->use_pair = p->precision == TCP_F32 && p->bc[0] == TCP_BC_PERIODIC && nx % 2 == 0;
    if (own) {
        void* mem = nullptr;
        e = cudaMalloc(&mem, s->L.total);
        if (e != cudaSuccess) { delete s; return cuda_fail(e, "cudaMalloc(workspace)"); }
        s->base = static_cast<char*>(mem);
        e = cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) { cudaFree(mem); delete s; return cuda_fail(e, "cudaStreamCreate"); }
    } else {
        if (!workspace) { delete s; return fail(TCP_EINVAL, "workspace is NULL"); }
        if (bytes < s->L.total) { delete s; return fail(TCP_EINVAL, "workspace smaller than tcp_workspace_bytes"); }
        if (reinterpret_cast<size_t>(workspace) % kAlign) { delete s; return fail(TCP_EINVAL, "workspace must be 256-byte aligned"); }
        s->base = static_cast<char*>(workspace);
        s->stream = static_cast<cudaStream_t>(stream);
    }
    if (cudaEventCreate(&s->ev0) != cudaSuccess || cudaEventCreate(&s->ev1) != cudaSuccess ||
        cudaEventCreate(&s->evc0) != cudaSuccess || cudaEventCreate(&s->evc1) != cudaSuccess ||
        cudaEventCreateWithFlags(&s->ev_bnd, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&s->ev_comm, cudaEventDisableTiming) != cudaSuccess) {
        tcp_destroy(s);
        return fail(TCP_ECUDA, "cudaEventCreate failed");
    }
    for (int a = 0; a < 3; ++a)
        for (int fc = 0; fc < 2; ++fc) {
            rc = p->precision == TCP_F64 ? fill_wall<double>(s, a, fc, nullptr) : fill_wall<float>(s, a, fc, nullptr);
            if (rc) { tcp_destroy(s); return rc; }
        }
    *out = s;
    return TCP_OK;
}

}  // namespace

extern "C" {

const char* tcp_last_error(void) { return g_err; }

int tcp_params_default(tcp_params* p) {
    if (!p) return fail(TCP_EINVAL, "params is NULL");
    std::memset(p, 0, sizeof *p);
    p->struct_size = sizeof(tcp_params);
    p->precision = TCP_F64; p->thermal = TCP_THERMAL_LB_D3Q7; p->streaming = TCP_STREAM_TWO_GRID;
    p->rho_H = p->rho_L = 1.0;
    p->tau_H = p->tau_L = 0.6;
    p->xi = 4.0; p->M = 0.05;
    p->kappa_H = p->kappa_L = 0.2;
    p->cp_H = p->cp_L = 1.0;
    p->s_bulk = p->s_high = 1.0;
    p->eps_normal = 1e-32;
    for (int a = 0; a < 3; ++a) p->wall_contact_angle[a][0] = p->wall_contact_angle[a][1] = 90.0;
    p->hydro_lattice = 27;
    return TCP_OK;
}

int tcp_workspace_bytes(int nx, int ny, int nz, const tcp_params* p, size_t* bytes) {
    if (!bytes) return fail(TCP_EINVAL, "bytes is NULL");
    int rc = validate(nx, ny, nz, p);
    if (rc) return rc;
    *bytes = make_layout(nx, ny, nz, p).total;
    return TCP_OK;
}

int tcp_create(int nx, int ny, int nz, const tcp_params* p, tcp_sim** out) {
    return create_common(nx, ny, nz, p, nullptr, 0, nullptr, true, out);
}

int tcp_create_in(int nx, int ny, int nz, const tcp_params* p, void* dev_workspace, size_t bytes, void* cuda_stream, tcp_sim** out) {
    return create_common(nx, ny, nz, p, dev_workspace, bytes, cuda_stream, false, out);
}

int tcp_destroy(tcp_sim* s) {
    if (!s) return TCP_OK;
    DeviceScope scope(s);
    cudaStreamSynchronize(s->stream);
    if (s->halo[0] || s->halo[1]) cudaStreamSynchronize(s->comm);
    if (s->ev0) cudaEventDestroy(s->ev0);
    if (s->ev1) cudaEventDestroy(s->ev1);
    if (s->evc0) cudaEventDestroy(s->evc0);
    if (s->evc1) cudaEventDestroy(s->evc1);
    if (s->ev_bnd) cudaEventDestroy(s->ev_bnd);
    if (s->ev_comm) cudaEventDestroy(s->ev_comm);
    if (s->owns_stream && s->stream) cudaStreamDestroy(s->stream);
    if (s->owns_memory && s->base) cudaFree(s->base);
    delete s;
    return TCP_OK;
}

int tcp_init_fields(tcp_sim* s, const void* phi, const void* u, const void* T) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    if (!phi) return fail(TCP_EINVAL, "phi is required");
    if (s->in_step) return fail(TCP_ESTATE, "tcp_init_fields between tcp_step_begin and tcp_step_end");
    DeviceScope scope(s);
    return s->P.precision == TCP_F64 ? init_fields_t<double>(s, phi, u, T) : init_fields_t<float>(s, phi, u, T);
}

int tcp_set_wall_temperature(tcp_sim* s, int axis, int face, const void* Tw) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    if (axis < 0 || axis > 2 || face < 0 || face > 1) return fail(TCP_EINVAL, "axis must be 0..2 and face 0..1");
    DeviceScope scope(s);
    return s->P.precision == TCP_F64 ? fill_wall<double>(s, axis, face, Tw) : fill_wall<float>(s, axis, face, Tw);
}

int tcp_set_heat_source(tcp_sim* s, const void* q) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    DeviceScope scope(s);
    s->has_q = q != nullptr;
    if (q) {
        const size_t es = s->P.precision == TCP_F64 ? 8 : 4;
        CK(cudaMemcpyAsync(s->base + s->L.q, q, s->N * es, cudaMemcpyDefault, s->stream));
        CK(cudaStreamSynchronize(s->stream));
    }
    return TCP_OK;
}

int tcp_step(tcp_sim* s, int nsteps) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    if (!s->initialised) return fail(TCP_ESTATE, "tcp_init_fields has not been called");
    if (nsteps < 0) return fail(TCP_EINVAL, "nsteps must be >= 0");
    if (s->halo[0] || s->halo[1]) return fail(TCP_ESTATE, "a slab with ghost planes steps with tcp_step_begin / tcp_step_end");
    DeviceScope scope(s);
    CK(cudaEventRecord(s->ev0, s->stream));
    for (int n = 0; n < nsteps; ++n) {
        int rc = s->P.precision == TCP_F64 ? step_once<double>(s) : step_once<float>(s);
        if (rc) return rc;
    }
    CK(cudaEventRecord(s->ev1, s->stream));
    CK(cudaGetLastError());
    s->stepped = true;
    return TCP_OK;
}

int tcp_relax_temperature(tcp_sim* s, int nsteps) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    if (!s->initialised) return fail(TCP_ESTATE, "tcp_init_fields has not been called");
    if (nsteps < 0) return fail(TCP_EINVAL, "nsteps must be >= 0");
    const bool lb = thermal_q(s->P.thermal) != 0;
    if (s->halo[0] || s->halo[1]) return fail(TCP_EUNSUPPORTED, "tcp_relax_temperature: not on a slab with ghost planes");
    if (lb && s->P.streaming == TCP_STREAM_AA && (nsteps & 1))
        return fail(TCP_EINVAL, "AA streaming: the thermal populations must keep the parity of h and g, so nsteps must be even");
    DeviceScope scope(s);
    return s->P.precision == TCP_F64 ? relax_t<double>(s, nsteps) : relax_t<float>(s, nsteps);
}

int tcp_read_fields(tcp_sim* s, void* phi, void* u, void* p, void* T) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    if (!s->initialised) return fail(TCP_ESTATE, "tcp_init_fields has not been called");
    DeviceScope scope(s);
    return s->P.precision == TCP_F64 ? read_fields_t<double>(s, phi, u, p, T) : read_fields_t<float>(s, phi, u, p, T);
}

int tcp_synchronize(tcp_sim* s) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    DeviceScope scope(s);
    CK(cudaStreamSynchronize(s->stream));
    CK(cudaGetLastError());
    return TCP_OK;
}

long long tcp_launch_count(const tcp_sim* s) { return s ? s->launches : 0; }

int tcp_halo_phases(const tcp_sim* s, int* phases) {
    if (!s || !phases) return fail(TCP_EINVAL, "NULL argument");
    *phases = halo_phases(s);
    return TCP_OK;
}

int tcp_halo_message_bytes(const tcp_sim* s, int phase, size_t* bytes) {
    if (!s || !bytes) return fail(TCP_EINVAL, "NULL argument");
    if (phase < 0 || phase >= halo_phases(s)) return fail(TCP_EINVAL, "phase out of range (tcp_halo_phases)");
    const int QT = thermal_q(s->P.thermal);
    const size_t planes = phase > 0 ? 1 : 9 + (size_t)tcp::halo_crossing(s->P.hydro_lattice, 1) + (size_t)tcp::halo_crossing(QT, 1) + 1 + (QT ? 1 : 0) + (rk_first_stage_fused(s) ? 1 : 0);
    *bytes = planes * s->nx * s->ny * (s->P.precision == TCP_F64 ? 8 : 4);
    return TCP_OK;
}

int tcp_halo_bytes(const tcp_sim* s, size_t* bytes) { return tcp_halo_message_bytes(s, 0, bytes); }

int tcp_set_halo(tcp_sim* s, int lo, int hi, void* comm_stream, void* send_lo, void* send_hi, void* recv_lo, void* recv_hi) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    if (s->in_step) return fail(TCP_ESTATE, "tcp_set_halo between tcp_step_begin and tcp_step_end");
    lo = lo != 0; hi = hi != 0;
    if (lo || hi) {
        if (s->P.streaming != TCP_STREAM_TWO_GRID) return fail(TCP_EUNSUPPORTED, "ghost planes: two-grid streaming only");
        if (s->nz - lo - hi < 1) return fail(TCP_EINVAL, "a slab needs at least one plane of its own between its ghost planes");
        if ((lo && (!send_lo || !recv_lo)) || (hi && (!send_hi || !recv_hi))) return fail(TCP_EINVAL, "a face with a ghost plane needs a send and a receive buffer");
    }
    s->halo[0] = lo; s->halo[1] = hi;
    s->comm = static_cast<cudaStream_t>(comm_stream);
    s->send[0] = send_lo; s->send[1] = send_hi; s->recv[0] = recv_lo; s->recv[1] = recv_hi;
    return TCP_OK;
}

int tcp_step_begin(tcp_sim* s) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    if (!s->initialised) return fail(TCP_ESTATE, "tcp_init_fields has not been called");
    if (!s->halo[0] && !s->halo[1]) return fail(TCP_ESTATE, "tcp_step_begin: no ghost planes (tcp_set_halo); use tcp_step");
    if (s->in_step) return fail(TCP_ESTATE, "tcp_step_begin called twice without tcp_step_end");
    DeviceScope scope(s);
    return s->P.precision == TCP_F64 ? step_begin_t<double>(s) : step_begin_t<float>(s);
}

int tcp_step_advance(tcp_sim* s, int* transfers_left) {
    if (!s || !transfers_left) return fail(TCP_EINVAL, "NULL argument");
    if (!s->in_step) return fail(TCP_ESTATE, "tcp_step_advance without tcp_step_begin");
    DeviceScope scope(s);
    return s->P.precision == TCP_F64 ? step_advance_t<double>(s, transfers_left) : step_advance_t<float>(s, transfers_left);
}

int tcp_step_end(tcp_sim* s) {
    if (!s) return fail(TCP_EINVAL, "sim is NULL");
    if (!s->in_step) return fail(TCP_ESTATE, "tcp_step_end without tcp_step_begin");
    if (s->phase + 1 < halo_phases(s)) return fail(TCP_ESTATE, "tcp_step_end: Runge-Kutta stages (and their transfers) are still to come, use tcp_step_advance");
    int left = 0;
    return tcp_step_advance(s, &left);
}

int tcp_read_pressure_static(tcp_sim* s, void* p) {
    if (!s || !p) return fail(TCP_EINVAL, "NULL argument");
    if (!s->initialised) return fail(TCP_ESTATE, "tcp_init_fields has not been called");
    if (s->in_step) return fail(TCP_ESTATE, "tcp_read_pressure_static between tcp_step_begin and tcp_step_end");
    const size_t es = s->P.precision == TCP_F64 ? 8 : 4;
    if (s->N * es > (size_t)TCP_STATIC_SCRATCH_BYTES)
        return fail(TCP_EUNSUPPORTED, "tcp_read_pressure_static: nx*ny*nz values exceed TCP_STATIC_SCRATCH_BYTES (8 MiB: 2^20 cells in fp64, 2^21 in fp32); use tcp_read_fields");
    DeviceScope scope(s);
    void*& scratch = g_static_scratch_addr[s->device];
    if (!scratch) {   // once per device, with that device current
        void* addr = nullptr;
        CK(cudaGetSymbolAddress(&addr, g_static_scratch));
        scratch = addr;
    }
    // every entry of [0, N) is written by the kernel before the copy reads it: the last call's contents never show
    if (s->P.precision == TCP_F64) launch_pressure<double>(s, static_cast<double*>(scratch));
    else launch_pressure<float>(s, static_cast<float*>(scratch));
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(p, scratch, s->N * es, cudaMemcpyDefault, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return TCP_OK;
}

int tcp_pattern_copy_ms(tcp_sim* s, int nlaunches, float* ms) {
    if (!s || !ms) return fail(TCP_EINVAL, "NULL argument");
    if (!s->initialised) return fail(TCP_ESTATE, "tcp_init_fields has not been called");
    if (nlaunches < 1) return fail(TCP_EINVAL, "nlaunches must be >= 1");
    if (s->walls || s->P.streaming != TCP_STREAM_TWO_GRID || s->halo[0] || s->halo[1] || s->P.hydro_lattice != 27)
        return fail(TCP_EUNSUPPORTED, "pattern copy: periodic two-grid simulations without ghost planes and with the D3Q27 hydrodynamic lattice only");
    DeviceScope scope(s);
    tcp::FusedCfg c;
    c.qt = thermal_q(s->P.thermal); c.walls = false; c.mode = 3; c.aa = 0; c.device = s->device; c.grid = grid_for(s->N);
    // its own events, and not counted by tcp_launch_count: the calibration is not part of the method
    CK(cudaEventRecord(s->evc0, s->stream));
    for (int i = 0; i < nlaunches; ++i) {
        // in -> out only: the simulation's current state (grid `cur`) is read, the spare grid is overwritten
        if (s->P.precision == TCP_F64) CK(tcp::launch_fused_periodic(c, make_args<double>(s), s->stream));
        else CK(tcp::launch_fused_periodic(c, make_args<float>(s), s->stream));
    }
    CK(cudaEventRecord(s->evc1, s->stream));
    CK(cudaEventSynchronize(s->evc1));
    float total = 0.f;
    CK(cudaEventElapsedTime(&total, s->evc0, s->evc1));
    *ms = total / nlaunches;
    return TCP_OK;
}

int tcp_last_step_ms(tcp_sim* s, float* ms) {
    if (!s || !ms) return fail(TCP_EINVAL, "NULL argument");
    if (!s->stepped) return fail(TCP_ESTATE, "tcp_step has not been called");
    DeviceScope scope(s);
    CK(cudaEventSynchronize(s->ev1));
    CK(cudaEventElapsedTime(ms, s->ev0, s->ev1));
    return TCP_OK;
}

}  // extern "C"
