// lbm_api.cu — context, launch layer and C ABI (include/lbm.h) of the B200-native LBM-LES path.
#include "../../include/lbm.h"
#include "lbm_core.cuh"
#include "lbm_setup.cuh"
#include "lbm_step.cuh"
#include "lbm_step_vec.cuh"
#include "lbm_inplace_launch.h"
#include "lbm_thermal.cuh"
#include "lbm_out.cuh"
#include "lbm_mesh.cuh"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#include <algorithm>

using namespace lbmk;

namespace {

constexpr size_t ALIGN = 256;
constexpr int MAX_MODES = LBM_MAX_INFLOW_MODES;
inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Halo-padded box (lbm_core.cuh): x pitch = nx + 2 rounded up to 32, ny + 2 rows, nz + 2 planes.
struct Layout {
    int px, py;
    long long Np, stride;
    size_t off_A, off_B, off_flags, off_links, off_fu, off_fum, off_modes, off_mean, off_damp, off_scratch, total;
    size_t fu_bytes;
    size_t scratch_bytes;
};

// precision: LBM_PREC_F32 / LBM_PREC_F64 / LBM_PREC_F32_S16 (include/lbm.h).  rs = bytes of the arithmetic type (side buffers,
// mean sums, tables), ss = bytes of a stored population, xoff = padded x of interior x = 0 (one 32-byte sector)
inline size_t real_bytes(int precision) { return precision == LBM_PREC_F64 ? 8 : 4; }
inline size_t store_bytes(int precision) { return precision == LBM_PREC_F64 ? 8 : (precision == LBM_PREC_F32_S16 ? 2 : 4); }
inline int xoff_of(int precision) { return precision == LBM_PREC_F32_S16 ? 16 : 8; }

Layout make_layout(int nx, int ny, int nz, int want_mean, int precision, int inplace = 0)
{
    Layout L{};
    const size_t rs = real_bytes(precision), ss = store_bytes(precision);
    L.px = (nx + xoff_of(precision) + 1 + 31) / 32 * 32;
    L.py = ny + 2;
    L.Np = (long long)L.px * L.py * (nz + 2);
    L.stride = (long long)align_up((size_t)L.Np, 64);
    size_t o = 0;
    L.off_A = o; o += align_up((size_t)Q * L.stride * ss, ALIGN);
    L.off_B = o; o += align_up((size_t)Q * L.stride * ss, ALIGN);
    if (inplace) { o = L.off_B; L.off_B = L.off_A; } // in-place streaming (lbm_inplace.cuh): one buffer serves as both
    L.off_flags = o; o += align_up((size_t)L.Np, ALIGN);
    L.off_links = o; o += align_up((size_t)L.Np * sizeof(uint32_t), ALIGN);
    // outflow-velocity side buffer (a6): 2 halves x 3 components x one slot per face-plane cell of all six faces (upper bound)
    L.fu_bytes = align_up((size_t)2 * 3 * 2 * ((size_t)ny * nz + (size_t)nx * nz + (size_t)nx * ny) * rs, ALIGN);
    L.off_fu = o; o += L.fu_bytes;
    // mean boundary velocity of the EQ slots (3 components) and the mode table of the synthetic inflow fluctuations
    L.off_fum = o; o += align_up(L.fu_bytes / 2, ALIGN);
    L.off_modes = o; o += align_up((size_t)MAX_MODES * 8 * sizeof(double), ALIGN);
    L.off_mean = o; if (want_mean) o += align_up((size_t)3 * L.stride * rs, ALIGN);
    // damping tables (lbm_set_damping): sx[nx], sy[ny], sz[nz], ut[3][nz]
    L.off_damp = o; o += align_up(((size_t)nx + ny + 4 * (size_t)nz) * rs, ALIGN);
    // scratch: heightmap (nx*ny int32) or a profile (3 nz doubles) or one face plane (3 n1 n2 doubles)
    const size_t plane = (size_t)std::max(std::max((size_t)nx * ny, (size_t)nx * nz), (size_t)ny * nz);
    L.scratch_bytes = align_up(std::max(plane * 3 * sizeof(double), (size_t)nz * 3 * sizeof(double)), ALIGN);
    L.off_scratch = o; o += L.scratch_bytes;
    L.total = o;
    return L;
}

// largest box: the padded cell count must fit a 32-bit int
bool size_ok(int nx, int ny, int nz)
{
    if (nx < 1 || ny < 1 || nz < 1 || nz > 65535) return false;
    const long long px = ((long long)nx + 16 + 1 + 31) / 32 * 32; // the widest row offset (16-bit storage)
    return px * ((long long)ny + 2) * ((long long)nz + 2) <= 2000000000LL;
}

} // namespace

struct lbm {
    int nx, ny, nz;
    double nu0, Cs, fv[3], F[3]; // fv = Coriolis vector f = 2 Omega; lbm_create's scalar f_cor is fv[2]
    int face[6];
    int fp64, s16, want_mean; // fp64: FP64 arithmetic and storage; s16: FP32 arithmetic, binary16 population storage
    int precision;            // LBM_PREC_* (without the streaming bit)
    int inplace;              // LBM_STREAM_INPLACE: one population buffer, cur = parity of the next step (lbm_inplace.cuh)
    int device;               // the CUDA device the handle was created on; every ABI call runs there (DevGuard)
    Layout L;
    char *ws;       // device workspace
    bool own_ws;
    cudaStream_t stream;
    int cur;        // which buffer holds the current state (0 = A, 1 = B)
    bool have_flags;
    long step;
    long mstart; int mevery; long mcount;
    long launches;
    int variant;
    bool damp_on;   // damping zones configured (the DAMP instantiation of the step kernel runs)
    int dlo[3], dhi[3]; // the zone-free inner box
    int nmodes;     // synthetic inflow fluctuations: modes in use (0 = off)
    bool thermal;   // D3Q7 thermal lattice + Boussinesq coupling on (lbm_set_thermal); its two buffers are library-owned
    double alpha, gbeta, theta_ref;
    int thd; double thw[6]; // fixed-temperature WALL faces (lbm_set_thermal_walls): mask and temperatures
    char *th_ws;    // [2][7][stride] reals + ft[2][F], cudaMalloc'ed by lbm_set_thermal, freed by lbm_destroy
    int loop_ok;    // multi-step cooperative launch: 0 = not probed yet, 1 = the whole grid is resident, -1 = no
    // staging buffers for HOST inputs / outputs that do not fit the scratch area (whole-lattice fields): kept between
    // calls, grown on demand, freed by lbm_destroy — a cudaMalloc + cudaFree pair per field per call costs milliseconds
    struct Slot { void *p; size_t cap; bool busy; } slots[4];
    std::string err;

    void *bufA() const { return ws + L.off_A; }
    void *bufB() const { return ws + L.off_B; }
    void *state() const { return cur ? bufB() : bufA(); }
    void *other() const { return cur ? bufA() : bufB(); }
    uint8_t *flags() const { return (uint8_t *)(ws + L.off_flags); }
    uint32_t *links() const { return (uint32_t *)(ws + L.off_links); }
    void *fu() const { return ws + L.off_fu; }
    void *mean() const { return want_mean ? ws + L.off_mean : nullptr; }
    void *fum() const { return ws + L.off_fum; }
    double *modes() const { return (double *)(ws + L.off_modes); }
    void *damp() const { return ws + L.off_damp; }
    void *scratch() const { return ws + L.off_scratch; }
    size_t pop_bytes() const { return (size_t)Q * (size_t)L.stride * (fp64 ? 8 : (s16 ? 2 : 4)); } // one population buffer
    size_t th_half() const { return (size_t)QT * (size_t)L.stride * (fp64 ? 8 : 4); }
    // thermal companion of the face-velocity side array: ft[2 halves][F] reals behind the two thermal buffers (F <= fu_bytes / 6 reals)
    size_t ft_bytes() const { return L.fu_bytes / 3; }
    char *ft() const { return th_ws + 2 * th_half(); }
    void *th_state() const { return thermal ? th_ws + (cur ? th_half() : 0) : nullptr; }
    void *th_other() const { return thermal ? th_ws + (cur ? 0 : th_half()) : nullptr; }
    long long N() const { return (long long)nx * ny * nz; }
};

namespace {

// Every ABI call runs on the handle's device whatever the caller's current device is, and restores the latter.
struct DevGuard {
    int prev = 0;
    bool sw = false;
    explicit DevGuard(const lbm_t *h)
    {
        if (!h) return;
        if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return; }
        sw = prev != h->device;
        if (sw) cudaSetDevice(h->device);
    }
    ~DevGuard() { if (sw) cudaSetDevice(prev); }
    DevGuard(const DevGuard &) = delete;
    DevGuard &operator=(const DevGuard &) = delete;
};

int fail(lbm_t *h, int code, const std::string &msg)
{
    if (h) h->err = msg;
    return code;
}

#define CUDA_TRY(h, expr)                                                                             \
    do {                                                                                              \
        cudaError_t e_ = (expr);                                                                      \
        if (e_ != cudaSuccess)                                                                        \
            return fail(h, LBM_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));            \
    } while (0)

// arithmetic type / storage type of a handle: <double, double>, <float, float> or <float, __half>
#define DISPATCH(h, fn, ...)                                                                            \
    ((h)->fp64 ? fn<double, double>(__VA_ARGS__) : ((h)->s16 ? fn<float, __half>(__VA_ARGS__) : fn<float, float>(__VA_ARGS__)))
#define DISPATCH_T(h, fn, T, ...)                                                                       \
    ((h)->fp64 ? fn<double, double, T>(__VA_ARGS__)                                                     \
               : ((h)->s16 ? fn<float, __half, T>(__VA_ARGS__) : fn<float, float, T>(__VA_ARGS__)))

template <typename real>
Params<real> make_params(const lbm_t *h)
{
    Params<real> P{};
    P.nx = h->nx; P.ny = h->ny; P.nz = h->nz;
    P.px = h->L.px; P.py = h->L.py; P.pxy = h->L.px * h->L.py;
    P.xoff = h->s16 ? 16 : 8; P.sec = h->s16 ? 16 : 8;
    P.perx = h->face[0] == LBM_PERIODIC ? 1 : 0; // set_boundaries guarantees both x faces then
    P.Np = (int)h->L.Np;
    P.N = (int)h->N();
    P.nxy = h->nx * h->ny;
    // exact for n < nxy + 1024 when (nxy + 1024) * nx < 2^32 (error term n * (magic * nx - 2^32) < 2^32)
    P.nx_magic = (h->nx > 1 && ((unsigned long long)P.nxy + 1024ULL) * (unsigned long long)h->nx < 0x100000000ULL)
                     ? (unsigned)((0x100000000ULL + (unsigned)h->nx - 1) / (unsigned)h->nx) : 0u;
    P.stride = h->L.stride;
    for (int k = 0; k < 6; ++k) P.face[k] = h->face[k];
    P.F = 0;
    for (int k = 0; k < 6; ++k) {
        const int axis = k >> 1;
        P.foff[k] = P.F;
        if (h->face[k] == FACE_EQ_OUTFLOW || h->face[k] == FACE_EQ_FIXED) P.F += (axis == 0 ? h->ny : h->nx) * (axis == 2 ? h->ny : h->nz);
    }
    P.tau0 = (real)(3.0 * h->nu0 + 0.5);
    P.Kles = (real)(18.0 * std::sqrt(2.0) * h->Cs * h->Cs);
    P.fx = (real)h->fv[0]; P.fy = (real)h->fv[1]; P.fz = (real)h->fv[2];
    P.hx = (real)(0.5 * h->fv[0]); P.hy = (real)(0.5 * h->fv[1]); P.hz = (real)(0.5 * h->fv[2]);
    P.inv1ph2 = (real)(1.0 / (1.0 + 0.25 * (h->fv[0] * h->fv[0] + h->fv[1] * h->fv[1] + h->fv[2] * h->fv[2])));
    P.Fx = (real)h->F[0]; P.Fy = (real)h->F[1]; P.Fz = (real)h->F[2];
    P.damp = h->damp_on ? (const real *)h->damp() : nullptr;
    for (int a = 0; a < 3; ++a) { P.dlo[a] = h->dlo[a]; P.dhi[a] = h->dhi[a]; }
    if (h->thermal) {
        P.gbeta = (real)h->gbeta; P.theta_ref = (real)h->theta_ref;
        P.omega_t = (real)(1.0 / (4.0 * h->alpha + 0.5));
        P.thd = h->thd;
        for (int k = 0; k < 6; ++k) P.thw[k] = (real)(2.0 * (h->thw[k] - h->theta_ref));
    }
    P.ipq = h->inplace ? h->cur : -1;
    return P;
}

inline unsigned blocks_for(long long n, int block) { return (unsigned)((n + block - 1) / block); }

// is p a device-accessible pointer? (device or managed memory)
bool is_device_ptr(const void *p)
{
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// Input staging.  Device sources are used in place; host sources are copied into the handle's scratch area when
// they fit at the given offset, else into a temporary allocation.  release_in waits for the copies (so that the
// caller's buffer is free on return) and frees temporaries.
constexpr size_t SLOT_MAX = (size_t)2 << 30; // larger requests are not cached
// a cached staging buffer of at least `bytes`; *slot = its index, or -1 for a one-off allocation (caller frees)
void *stage_alloc(lbm_t *h, size_t bytes, int *slot)
{
    *slot = -1;
    if (bytes <= SLOT_MAX) {
        int pick = -1;
        for (int k = 0; k < 4; ++k)
            if (!h->slots[k].busy && h->slots[k].cap >= bytes && (pick < 0 || h->slots[k].cap < h->slots[pick].cap)) pick = k;
        if (pick < 0)
            for (int k = 0; k < 4; ++k)
                if (!h->slots[k].busy && (pick < 0 || h->slots[k].cap < h->slots[pick].cap)) pick = k;
        if (pick >= 0) {
            lbm::Slot &s = h->slots[pick];
            if (s.cap < bytes) {
                if (s.p) cudaFree(s.p);
                s.p = nullptr; s.cap = 0;
                if (cudaMalloc(&s.p, bytes) != cudaSuccess) { cudaGetLastError(); s.p = nullptr; return nullptr; }
                s.cap = bytes;
            }
            s.busy = true;
            *slot = pick;
            return s.p;
        }
    }
    void *d = nullptr;
    if (cudaMalloc(&d, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return d;
}
void stage_free(lbm_t *h, void *p, int slot)
{
    if (slot >= 0) h->slots[slot].busy = false;
    else if (p) cudaFree(p);
}

struct InBuf { const void *dev; void *tmp; bool host; int slot; };
int stage_in(lbm_t *h, const void *src, size_t bytes, size_t scratch_off, InBuf *b)
{
    b->dev = nullptr; b->tmp = nullptr; b->host = false; b->slot = -1;
    if (!src) return LBM_OK;
    if (is_device_ptr(src)) { b->dev = src; return LBM_OK; }
    void *d = nullptr;
    if (scratch_off + bytes <= h->L.scratch_bytes) d = (char *)h->scratch() + scratch_off;
    else {
        d = stage_alloc(h, bytes, &b->slot);
        if (!d) return fail(h, LBM_ENOMEM, "cudaMalloc staging (input)");
        b->tmp = d;
    }
    cudaError_t e = cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, h->stream);
    if (e != cudaSuccess) {
        if (b->tmp) stage_free(h, b->tmp, b->slot);
        b->tmp = nullptr;
        return fail(h, LBM_ECUDA, std::string("H2D copy: ") + cudaGetErrorString(e));
    }
    b->dev = d; b->host = true;
    return LBM_OK;
}
void release_in(lbm_t *h, InBuf *b, int n)
{
    bool any = false;
    for (int k = 0; k < n; ++k) any |= b[k].host;
    if (any) cudaStreamSynchronize(h->stream);
    for (int k = 0; k < n; ++k)
        if (b[k].tmp) { stage_free(h, b[k].tmp, b[k].slot); b[k].tmp = nullptr; }
}

// Output staging: if dst is a host pointer allocate a device buffer; finish_out copies back and frees.
struct OutBuf { void *host; void *dev; size_t bytes; bool temp; int slot; };
int stage_out(lbm_t *h, void *dst, size_t bytes, OutBuf *o)
{
    o->host = nullptr; o->dev = nullptr; o->bytes = bytes; o->temp = false; o->slot = -1;
    if (!dst) return LBM_OK;
    if (is_device_ptr(dst)) { o->dev = dst; return LBM_OK; }
    o->dev = stage_alloc(h, bytes, &o->slot);
    if (!o->dev) return fail(h, LBM_ENOMEM, "cudaMalloc staging (output)");
    o->host = dst; o->temp = true;
    return LBM_OK;
}
int finish_out(lbm_t *h, OutBuf *outs, int n)
{
    int rc = LBM_OK;
    bool any_host = false;
    for (int k = 0; k < n; ++k)
        if (outs[k].temp) {
            any_host = true;
            cudaError_t e = cudaMemcpyAsync(outs[k].host, outs[k].dev, outs[k].bytes, cudaMemcpyDeviceToHost, h->stream);
            if (e != cudaSuccess) rc = fail(h, LBM_ECUDA, std::string("D2H copy: ") + cudaGetErrorString(e));
        }
    if (any_host) {
        cudaError_t e = cudaStreamSynchronize(h->stream);
        if (e != cudaSuccess) rc = fail(h, LBM_ECUDA, std::string("sync: ") + cudaGetErrorString(e));
    }
    for (int k = 0; k < n; ++k)
        if (outs[k].temp) stage_free(h, outs[k].dev, outs[k].slot);
    return rc;
}

int check_launch(lbm_t *h, const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, LBM_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
    h->launches += 1;
    return LBM_OK;
}

// ---- templated implementations -----------------------------------------------------------------------------------

template <typename real, typename S>
int do_set_flags(lbm_t *h, const int32_t *height, const uint8_t *dev_mask = nullptr, int thresh = 1)
{
    const Params<real> P = make_params<real>(h);
    InBuf in;
    int rc = stage_in(h, height, (size_t)h->nx * h->ny * sizeof(int32_t), 0, &in);
    if (rc) return rc;
    const int B = 256;
    voxelise_kernel<real><<<blocks_for(P.Np, B), B, 0, h->stream>>>((const int32_t *)in.dev, dev_mask, thresh, h->flags(), P);
    rc = check_launch(h, "voxelise_kernel");
    if (!rc) {
        rc = cudaMemsetAsync(h->links(), 0, (size_t)P.Np * sizeof(uint32_t), h->stream) == cudaSuccess ? LBM_OK
             : fail(h, LBM_ECUDA, "memset links");
    }
    if (!rc) {
        // in place: class bits are never changed by classify, only the SLOW / EDGE bits are added
        const dim3 cg((unsigned)(P.px / CT_X), blocks_for(P.ny, CT_Y), blocks_for(P.nz, CT_Z));
        if (cg.y <= 65535u && cg.z <= 65535u) // tiled through shared memory; very flat / long boxes beyond the grid limits: one thread per cell
            classify_tiled_kernel<real><<<cg, dim3(CT_X, CT_Y, CT_Z), 0, h->stream>>>(h->flags(), h->links(), P);
        else
            classify_kernel<real><<<blocks_for(P.N, B), B, 0, h->stream>>>(h->flags(), h->links(), P);
        rc = check_launch(h, "classify_kernel");
    }
    release_in(h, &in, 1);
    if (rc) return rc;
    const size_t rs = sizeof(real);
    CUDA_TRY(h, cudaMemsetAsync(h->bufA(), 0, h->pop_bytes(), h->stream));
    if (!h->inplace) CUDA_TRY(h, cudaMemsetAsync(h->bufB(), 0, h->pop_bytes(), h->stream));
    if (h->want_mean) CUDA_TRY(h, cudaMemsetAsync(h->mean(), 0, (size_t)3 * h->L.stride * rs, h->stream));
    CUDA_TRY(h, cudaMemsetAsync(h->fu(), 0, h->L.fu_bytes, h->stream));
    if (h->thermal) CUDA_TRY(h, cudaMemsetAsync(h->ft(), 0, h->ft_bytes(), h->stream)); // theta_b back to theta_ref; the thermal state is stale until lbm_set_theta
    h->cur = 0; h->step = 0; h->mcount = 0; h->have_flags = true;
    return LBM_OK;
}

template <typename real, typename in_t>
int do_inlet_theta(lbm_t *h, const in_t *theta_b);
// the boundary velocity changed while the thermal lattice is on: the EQ_FIXED cells' thermal state h_eq(theta_b, u_b) follows
template <typename real>
int thermal_refresh(lbm_t *h) { return h->thermal ? do_inlet_theta<real, float>(h, nullptr) : LBM_OK; }

template <typename real, typename S, typename in_t>
int do_set_inlet(lbm_t *h, int mode, int face, const in_t *u, const in_t *v, const in_t *w, size_t count)
{
    if (!h->have_flags) return fail(h, LBM_ESTATE, "set_inlet: flags not set");
    if (h->nmodes > 0) return fail(h, LBM_ESTATE, "set_inlet: the mean boundary state is fixed while inflow fluctuations are on");
    if (!u) return fail(h, LBM_EINVAL, "set_inlet: u is NULL");
    const Params<real> P = make_params<real>(h);
    InBuf in[3];
    const size_t bytes = count * sizeof(in_t);
    int rc = stage_in(h, u, bytes, 0, &in[0]);
    if (!rc) rc = stage_in(h, v, bytes, align_up(bytes, ALIGN), &in[1]); else in[1] = InBuf{nullptr, nullptr, false, -1};
    if (!rc) rc = stage_in(h, w, bytes, 2 * align_up(bytes, ALIGN), &in[2]); else in[2] = InBuf{nullptr, nullptr, false, -1};
    if (!rc) {
        const int B = 256;
        const long long threads = mode == 0 ? (long long)std::max(P.F, 1) : (long long)count;
        inlet_kernel<real, S, in_t><<<blocks_for(threads, B), B, 0, h->stream>>>(
            (S *)h->bufA(), (S *)h->bufB(), (real *)h->fu(), h->flags(), (const in_t *)in[0].dev, (const in_t *)in[1].dev,
            (const in_t *)in[2].dev, mode, face, P);
        rc = check_launch(h, "inlet_kernel");
        if (!rc) rc = thermal_refresh<real>(h);
    }
    release_in(h, in, 3);
    return rc;
}

template <typename in_t>
int set_inlet_profile_any(lbm_t *h, const in_t *u, const in_t *v, const in_t *w)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    return DISPATCH_T(h, do_set_inlet, in_t, h, 0, 0, u, v, w, (size_t)h->nz);
}

template <typename in_t>
int set_inlet_plane_any(lbm_t *h, int face, const in_t *uvw)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (face < 0 || face > 5) return fail(h, LBM_EINVAL, "set_inlet_plane: face out of range");
    if (!uvw) return fail(h, LBM_EINVAL, "set_inlet_plane: uvw is NULL");
    const int axis = face / 2;
    const size_t n1 = axis == 0 ? h->ny : h->nx, n2 = axis == 2 ? h->ny : h->nz;
    const size_t cnt = n1 * n2;
    // stage the three planes as one array so that a host source is copied once (it fits the scratch area)
    InBuf in;
    int rc = stage_in(h, uvw, 3 * cnt * sizeof(in_t), 0, &in);
    if (rc) return rc;
    const in_t *p = (const in_t *)in.dev;
    rc = DISPATCH_T(h, do_set_inlet, in_t, h, 1, face, p, p + cnt, p + 2 * cnt, cnt);
    release_in(h, &in, 1);
    return rc;
}

template <typename real, typename S>
int do_fluct(lbm_t *h, double t, bool cells);

// Mesh voxeliser (lbm_mesh.cuh): vote counts of the three ray passes, in the first N bytes of the link-word area (free
// until classify_kernel rewrites it); the toggles of the running pass sit in the bytes behind them.
int mesh_votes(lbm_t *h, int n_tri, const float *dev_tri, uint8_t **votes_out)
{
    const long long N = h->N();
    uint8_t *votes = (uint8_t *)h->links();
    const size_t tog_off = align_up((size_t)N, ALIGN), tog_bytes = align_up((size_t)N, 4) + 4;
    uint8_t *toggles = votes + tog_off;
    int *err = (int *)(toggles + align_up(tog_bytes, ALIGN));
    // 4 Np bytes are there: N votes + N toggles + a flag word fit for every box (Np >= N + halo)
    if (tog_off + align_up(tog_bytes, ALIGN) + sizeof(int) > (size_t)h->L.Np * sizeof(uint32_t))
        return fail(h, LBM_ENOMEM, "set_flags_mesh: box too small for the scratch layout");
    CUDA_TRY(h, cudaMemsetAsync(votes, 0, (size_t)N, h->stream));
    CUDA_TRY(h, cudaMemsetAsync(err, 0, sizeof(int), h->stream));
    const int B = 128;
    const unsigned tg = blocks_for((long long)n_tri * 32, B);
    const int n[3] = {h->nx, h->ny, h->nz};
    for (int d = 0; d < 3 && n_tri > 0; ++d) {
        CUDA_TRY(h, cudaMemsetAsync(toggles, 0, tog_bytes, h->stream));
        const unsigned sg = blocks_for((long long)n[(d + 1) % 3] * n[(d + 2) % 3], B);
        if (d == 0) {
            mesh_toggle_kernel<0><<<tg, B, 0, h->stream>>>(dev_tri, n_tri, (uint32_t *)toggles, h->nx, h->ny, h->nz, err);
            mesh_scan_kernel<0><<<sg, B, 0, h->stream>>>(toggles, votes, h->nx, h->ny, h->nz);
        } else if (d == 1) {
            mesh_toggle_kernel<1><<<tg, B, 0, h->stream>>>(dev_tri, n_tri, (uint32_t *)toggles, h->nx, h->ny, h->nz, err);
            mesh_scan_kernel<1><<<sg, B, 0, h->stream>>>(toggles, votes, h->nx, h->ny, h->nz);
        } else {
            mesh_toggle_kernel<2><<<tg, B, 0, h->stream>>>(dev_tri, n_tri, (uint32_t *)toggles, h->nx, h->ny, h->nz, err);
            mesh_scan_kernel<2><<<sg, B, 0, h->stream>>>(toggles, votes, h->nx, h->ny, h->nz);
        }
        int rc = check_launch(h, "mesh_toggle_kernel / mesh_scan_kernel");
        if (rc) return rc;
        h->launches += 1;
    }
    int bad = 0;
    CUDA_TRY(h, cudaMemcpyAsync(&bad, err, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (bad) return fail(h, LBM_EINVAL, "set_flags_mesh: a vertex is not finite or outside [-1024, 2048) cells");
    *votes_out = votes;
    return LBM_OK;
}
template <typename real, typename S>
int turb_publish(lbm_t *h, bool cells);

template <typename real, typename S, typename in_t>
int do_set_macros(lbm_t *h, const in_t *rho, const in_t *ux, const in_t *uy, const in_t *uz)
{
    if (!h->have_flags) return fail(h, LBM_ESTATE, "set_macros: flags not set");
    const Params<real> P = make_params<real>(h);
    const size_t bytes = (size_t)P.N * sizeof(in_t);
    InBuf in[4] = {};
    const in_t *src[4] = {rho, ux, uy, uz};
    int rc = LBM_OK;
    for (int k = 0; k < 4 && !rc; ++k) rc = stage_in(h, src[k], bytes, h->L.scratch_bytes, &in[k]); // never fits: temp
    if (!rc) {
        const int B = 256;
        if (h->inplace)
            init_kernel<real, S, in_t, 1><<<blocks_for(P.N, B), B, 0, h->stream>>>(
                (S *)h->bufA(), (S *)nullptr, (real *)h->fu(), h->flags(), h->links(), (const in_t *)in[0].dev, (const in_t *)in[1].dev,
                (const in_t *)in[2].dev, (const in_t *)in[3].dev, P);
        else
            init_kernel<real, S, in_t, 0><<<blocks_for(P.N, B), B, 0, h->stream>>>(
                (S *)h->bufA(), (S *)nullptr, (real *)h->fu(), h->flags(), h->links(), (const in_t *)in[0].dev, (const in_t *)in[1].dev,
                (const in_t *)in[2].dev, (const in_t *)in[3].dev, P);
        rc = check_launch(h, "init_kernel");
    }
    release_in(h, in, 4);
    if (!rc) { h->step = 0; if (!h->inplace) h->cur = 0; } // in-place streaming: written in the layout of the current parity
    if (!rc && h->nmodes > 0) rc = turb_publish<real, S>(h, true); // the step counter restarts: the inflow cells carry u'(x, 0)
    return rc;
}

template <typename real, typename S, bool SPEC, int BLOCK, int MINB, bool DAMP = false, bool TURB = false, bool PERX = false>
int launch_step_as(lbm_t *h, const Params<real> &P, bool sample)
{
    if constexpr (!PERX) {
        // the read-side wrap instantiation carries two more cell indices: one CTA per SM less instead of spills
        if (P.perx) return launch_step_as<real, S, SPEC, BLOCK, (SPEC && MINB == 10) ? 9 : MINB, DAMP, TURB, true>(h, P, sample);
    }
    const S *A = (const S *)h->state();
    S *B = (S *)h->other();
    real *ms = (real *)h->mean();
    dim3 grid(blocks_for((long long)P.nxy, BLOCK), (unsigned)P.nz);
    // TURB: leading block rows that carry the face slots; they publish the boundary velocity of step (this one) + 1
    const int turb_planes = TURB ? (int)((blocks_for(P.F, BLOCK) + grid.x - 1) / grid.x) : 0;
    grid.y += turb_planes;
    const Turb<real> tb{(const real *)h->fum(), h->modes(), h->nmodes, (double)(h->step + 2)};
    const StepPtrs<S> T = make_step_ptrs<S>(A, B, P);
    // the side buffer's halves follow the population buffers: read the half written together with A, write B's
    const real *fur = (const real *)h->fu() + (size_t)(h->cur ? 3 : 0) * P.F;
    real *fuw = (real *)h->fu() + (size_t)(h->cur ? 0 : 3) * P.F;
    // sampling steps hold three more values per thread (the prefetched sums): one CTA per SM less, 56 registers, no spills
    constexpr int MINB_S = (SPEC && MINB == 10) ? 9 : MINB;
    // Programmatic dependent launch (lbm_step.cuh): back-to-back steps overlap the next launch's set-up and index arithmetic with
    // the drain of the running one; the kernel touches no memory before griddepcontrol.wait.  Measured: config 2 (65 us per
    // step) +2.6 %, config 3 +0.5 %, config 1 with one launch per step +7 %.
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = dim3(BLOCK); cfg.dynamicSmemBytes = 0; cfg.stream = h->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    const uint8_t *fl = h->flags();
    const uint32_t *lk = h->links();
    if (sample) cudaLaunchKernelEx(&cfg, step_kernel<real, S, true, SPEC, BLOCK, MINB_S, DAMP, TURB, PERX>, A, B, fl, lk, ms, fur, fuw, P, T, tb, turb_planes);
    else cudaLaunchKernelEx(&cfg, step_kernel<real, S, false, SPEC, BLOCK, MINB, DAMP, TURB, PERX>, A, B, fl, lk, ms, fur, fuw, P, T, tb, turb_planes);
    return check_launch(h, "step_kernel");
}

// V cells per thread, 64/128-bit accesses (lbm_step_vec.cuh); applicable when nx % V == 0 and the thread index divides exactly
template <int V>
bool vec_geom(const Params<float> &P, VecGeom *G)
{
    if (P.nx % V != 0 || P.perx) return false; // periodic x: the read-side wrap lives in the one-cell kernel only
    G->qpr = (unsigned)(P.nx / V);
    G->nq = (unsigned)((long long)P.nxy / V);
    G->qmagic = 0;
    // exact for n < nq + 1024 when (nq + 1024) * qpr < 2^32 (error term n * (magic * qpr - 2^32) < 2^32)
    if (G->qpr > 1 && ((unsigned long long)G->nq + 1024ULL) * G->qpr < 0x100000000ULL)
        G->qmagic = (unsigned)((0x100000000ULL + G->qpr - 1) / G->qpr);
    return true;
}
template <typename S, int V, int MINB, int MINB_S>
int launch_step_vec(lbm_t *h, const Params<float> &P, const VecGeom &G, bool sample)
{
    constexpr int BLOCK = 128;
    const S *A = (const S *)h->state();
    S *B = (S *)h->other();
    const dim3 grid(blocks_for((long long)G.nq, BLOCK), (unsigned)P.nz);
    const VecPtrs<S> T = make_vec_ptrs<S>(A, B, P);
    const float *fur = (const float *)h->fu() + (size_t)(h->cur ? 3 : 0) * P.F;
    float *fuw = (float *)h->fu() + (size_t)(h->cur ? 0 : 3) * P.F;
    if (sample) step_vec_kernel<S, V, true, BLOCK, MINB_S><<<grid, BLOCK, 0, h->stream>>>(h->flags(), h->links(), (float *)h->mean(), fur, fuw, P, T, G);
    else step_vec_kernel<S, V, false, BLOCK, MINB><<<grid, BLOCK, 0, h->stream>>>(h->flags(), h->links(), nullptr, fur, fuw, P, T, G);
    return check_launch(h, "step_vec_kernel");
}

// launch shapes of the FP32 step (lbm_set_variant): the same arithmetic and the same stored state in all of them
//   0 = default: one cell per thread; lattices whose whole grid is resident at once run several steps per cooperative
//       launch (step_loop_kernel)
//   1 = one cell per thread, one launch per step
//   2 = 2 cells per thread with 64-bit accesses (16-bit storage: 32-bit) where nx % 2 == 0, else as 1
//   3 = 4 cells per thread with 128-bit accesses (16-bit storage: 64-bit) where nx % 4 == 0, else as 1
constexpr int N_VARIANTS = 4;
#ifndef DAMP_MINB
#define DAMP_MINB 9
#endif
#ifndef THERMAL_MINB
#define THERMAL_MINB 9
#endif
#ifndef VEC4_MINB
#define VEC4_MINB 4
#endif
#ifndef VEC2_MINB
#define VEC2_MINB 6
#endif
// in-place streaming (lbm_inplace.cuh; kernels and launch in lbm_inplace_launch.cu): one launch shape, one cell per thread;
// cur = parity of this step
template <typename real, typename S>
int launch_ip_step(lbm_t *h, const Params<real> &P, bool sample)
{
    IpLaunch L{};
    L.prec = h->fp64 ? 1 : (h->s16 ? 2 : 0);
    L.sample = sample; L.damp = h->damp_on; L.turb = h->nmodes > 0 && P.F > 0;
    L.parity = h->cur;
    L.G = h->bufA(); L.flags = h->flags(); L.links = h->links(); L.msum = h->mean();
    // the side buffer's halves follow the parity as they follow the buffers of the two-buffer scheme
    L.fur = (const real *)h->fu() + (size_t)(h->cur ? 3 : 0) * P.F;
    L.fuw = (real *)h->fu() + (size_t)(h->cur ? 0 : 3) * P.F;
    L.params = &P;
    L.fum = h->fum(); L.modes = h->modes(); L.nmodes = h->nmodes; L.t = (double)(h->step + 2);
    if (h->thermal) { // the thermal populations stay double-buffered; their halves follow the parity as the side arrays do
        real *ft = (real *)h->ft();
        L.HA = h->th_state(); L.HB = h->th_other();
        L.ftr = ft + (size_t)(h->cur ? 1 : 0) * P.F; L.ftw = ft + (size_t)(h->cur ? 0 : 1) * P.F;
    }
    L.stream = h->stream;
    ip_launch(L);
    return check_launch(h, h->thermal ? "ip_thermal_step_kernel" : "ip_step_kernel");
}

template <typename real, typename S>
int launch_step(lbm_t *h, const Params<real> &P, bool sample)
{
    if (h->inplace) return launch_ip_step<real, S>(h, P, sample);
    if (h->thermal) { // fused flow + thermal step (lbm_thermal.cuh); S = real there (lbm_set_thermal refuses 16-bit storage)
        const real *A = (const real *)h->state();
        real *B = (real *)h->other();
        dim3 grid(blocks_for((long long)P.nxy, 128), (unsigned)P.nz);
        // 19 + 7 populations.  With the buoyancy passed into collide() as a value (P stays in the constant bank) and the address
        // table, 56 registers (9 CTAs per SM, 16 B of spills) measure best: 26 030 MLUPS against 25 860 at 8 CTAs (64 registers, no
        // spills), 24 450 at 10 CTAs (48 registers, 108 B of spills) and round 1's 24 600 at 7 CTAs (72 registers)
        constexpr int BLOCK = 128, MINB = std::is_same<real, float>::value ? THERMAL_MINB : 2;
        const ThermalPtrs<real> T = make_thermal_ptrs<real>(A, B, (const real *)h->th_state(), (real *)h->th_other(), P);
        // the side arrays' halves follow the population buffers (as in launch_step_as)
        real *fu = (real *)h->fu(), *ft = (real *)h->ft();
        const OpenFaces<real> O{fu + (size_t)(h->cur ? 3 : 0) * P.F, fu + (size_t)(h->cur ? 0 : 3) * P.F, ft + (size_t)(h->cur ? 1 : 0) * P.F,
                                ft + (size_t)(h->cur ? 0 : 1) * P.F};
        cudaLaunchConfig_t cfg{}; // programmatic dependent launch, as for the plain step (launch_step_as)
        cfg.gridDim = grid; cfg.blockDim = dim3(BLOCK); cfg.dynamicSmemBytes = 0; cfg.stream = h->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        real *HB = (real *)h->th_other(), *msum = (real *)h->mean();
        const uint8_t *fl = h->flags();
        const uint32_t *lk = h->links();
        const bool turb = h->nmodes > 0 && P.F > 0;
        if (h->damp_on || turb) { // damping zones / inflow fluctuations together with the thermal lattice: their own instantiation (one CTA per SM less)
            constexpr int MD = std::is_same<real, float>::value ? (MINB > 8 ? 8 : MINB) : MINB;
            // leading block rows that carry the face slots; they publish the boundary velocity of step (this one) + 1 (launch_step_as)
            const int turb_planes = turb ? (int)((blocks_for(P.F, BLOCK) + grid.x - 1) / grid.x) : 0;
            cfg.gridDim.y += turb_planes;
            const Turb<real> tb{(const real *)h->fum(), h->modes(), h->nmodes, (double)(h->step + 2)};
            if (P.perx) {
                if (sample) cudaLaunchKernelEx(&cfg, thermal_step_kernel<real, true, BLOCK, MD, true, true>, B, HB, fl, lk, msum, P, T, O, tb, turb_planes);
                else cudaLaunchKernelEx(&cfg, thermal_step_kernel<real, false, BLOCK, MD, true, true>, B, HB, fl, lk, msum, P, T, O, tb, turb_planes);
            } else {
                if (sample) cudaLaunchKernelEx(&cfg, thermal_step_kernel<real, true, BLOCK, MD, false, true>, B, HB, fl, lk, msum, P, T, O, tb, turb_planes);
                else cudaLaunchKernelEx(&cfg, thermal_step_kernel<real, false, BLOCK, MD, false, true>, B, HB, fl, lk, msum, P, T, O, tb, turb_planes);
            }
        } else if (P.perx) {
            if (sample) cudaLaunchKernelEx(&cfg, thermal_step_kernel<real, true, BLOCK, MINB, true>, B, HB, fl, lk, msum, P, T, O, Turb<real>{}, 0);
            else cudaLaunchKernelEx(&cfg, thermal_step_kernel<real, false, BLOCK, MINB, true>, B, HB, fl, lk, msum, P, T, O, Turb<real>{}, 0);
        } else {
            if (sample) cudaLaunchKernelEx(&cfg, thermal_step_kernel<real, true, BLOCK, MINB, false>, B, HB, fl, lk, msum, P, T, O, Turb<real>{}, 0);
            else cudaLaunchKernelEx(&cfg, thermal_step_kernel<real, false, BLOCK, MINB, false>, B, HB, fl, lk, msum, P, T, O, Turb<real>{}, 0);
        }
        return check_launch(h, "thermal_step_kernel");
    }
    const bool turb = h->nmodes > 0 && P.F > 0;
    if (h->damp_on || turb) { // damping zones / inflow fluctuations: their own instantiations (same arithmetic elsewhere)
        if constexpr (std::is_same<real, float>::value) {
            if (h->damp_on && turb) return launch_step_as<real, S, true, 128, DAMP_MINB, true, true>(h, P, sample);
            if (h->damp_on) return launch_step_as<real, S, true, 128, DAMP_MINB, true, false>(h, P, sample);
            return launch_step_as<real, S, true, 128, 10, false, true>(h, P, sample); // no prefetched table values: 48 registers do
        } else {
            if (h->damp_on && turb) return launch_step_as<real, S, false, 256, 2, true, true>(h, P, sample);
            if (h->damp_on) return launch_step_as<real, S, false, 256, 2, true, false>(h, P, sample);
            return launch_step_as<real, S, false, 256, 2, false, true>(h, P, sample);
        }
    }
    if constexpr (std::is_same<real, float>::value) {
        VecGeom G;
        if (h->variant == 3 && vec_geom<4>(P, &G)) return launch_step_vec<S, 4, VEC4_MINB, 3>(h, P, G, sample);
        if constexpr (std::is_same<S, float>::value) {
            if (h->variant == 2 && vec_geom<2>(P, &G)) return launch_step_vec<S, 2, VEC2_MINB, 5>(h, P, G, sample);
        } else {
            if (h->variant == 2 && vec_geom<2>(P, &G)) return launch_step_vec<S, 2, VEC2_MINB, 5>(h, P, G, sample);
        }
        return launch_step_as<real, S, true, 128, 10>(h, P, sample);
    } else return launch_step_as<real, S, false, 256, 2>(h, P, sample);
}

// boundary velocities of time t for the EQ_FIXED slots (mean + fluctuations on active inflow cells); cells = also rewrite
// the cells' populations (set-up / switch-off / re-initialisation)
template <typename real, typename S>
int do_fluct(lbm_t *h, double t, bool cells)
{
    const Params<real> P = make_params<real>(h);
    if (P.F == 0) return LBM_OK;
    const int B = 128;
    const Turb<real> tb{(const real *)h->fum(), h->modes(), h->nmodes, t};
    if (cells) fluct_kernel<real, S, true><<<blocks_for(P.F, B), B, 0, h->stream>>>((S *)h->bufA(), (S *)h->bufB(), (real *)h->fu(), h->flags(), tb, P);
    else fluct_kernel<real, S, false><<<blocks_for(P.F, B), B, 0, h->stream>>>((S *)nullptr, (S *)nullptr, (real *)h->fu(), h->flags(), tb, P);
    return check_launch(h, "fluct_kernel");
}

// Fluctuations on: the EQ_FIXED cells hold u_b(step) and both halves of the side array u_b(step + 1), which the next
// launch re-expands; from then on every launch publishes the velocity of the step after its own (TURB blocks).
template <typename real, typename S>
int turb_publish(lbm_t *h, bool cells)
{
    int rc = cells ? do_fluct<real, S>(h, (double)h->step, true) : LBM_OK;
    // the cells now hold f_eq(1, u_b(step)) and the side array that velocity: their thermal state follows it (reading 28) ...
    if (!rc && cells) rc = thermal_refresh<real>(h);
    // ... before the side array moves on to u_b(step + 1), which the next launch re-expands
    if (!rc) rc = do_fluct<real, S>(h, (double)(h->step + 1), false);
    return rc;
}

// Small lattices (the whole grid resident at once): 2 * pairs steps in one cooperative launch (step_loop_kernel).
// Returns the number of steps done (0 = not applicable here: use single launches), or a negative error code.
template <typename real, typename S>
int try_step_loop(lbm_t *h, const Params<real> &P, int want)
{
    if constexpr (!std::is_same<real, float>::value) return 0;
    else {
        if (h->variant != 0 || h->nmodes > 0 || h->thermal || h->inplace || want < 4 || h->loop_ok < 0) return 0;
        constexpr int BLOCK = 128;
        const dim3 grid(blocks_for((long long)P.nxy, BLOCK), (unsigned)P.nz);
        const void *fn = P.perx ? (h->damp_on ? (const void *)step_loop_kernel<float, S, BLOCK, 8, true, true> : (const void *)step_loop_kernel<float, S, BLOCK, 8, false, true>)
                                : (h->damp_on ? (const void *)step_loop_kernel<float, S, BLOCK, 8, true, false> : (const void *)step_loop_kernel<float, S, BLOCK, 8, false, false>);
        if (h->loop_ok == 0) { // once per handle: can the whole grid be resident?
            int dev = 0, sms = 0, coop = 0, per_sm = 0;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, BLOCK, 0);
            h->loop_ok = (coop && (long long)per_sm * sms >= (long long)grid.x * grid.y) ? 1 : -1;
            cudaGetLastError();
            if (h->loop_ok < 0) return 0;
        }
        int pairs = want / 2;
        S *A = (S *)h->state(), *B = (S *)h->other();
        real *fu0 = (real *)h->fu() + (size_t)(h->cur ? 3 : 0) * P.F, *fu1 = (real *)h->fu() + (size_t)(h->cur ? 0 : 3) * P.F;
        StepPtrs<S> T0 = make_step_ptrs<S>(A, B, P), T1 = make_step_ptrs<S>(B, A, P);
        const uint8_t *fl = h->flags();
        const uint32_t *lk = h->links();
        Params<real> Pc = P;
        void *args[] = {&A, &B, &fl, &lk, &fu0, &fu1, &Pc, &T0, &T1, &pairs};
        cudaError_t e = cudaLaunchCooperativeKernel(fn, grid, dim3(BLOCK), args, 0, h->stream);
        if (e != cudaSuccess) { cudaGetLastError(); h->loop_ok = -1; return 0; } // e.g. too large after all: single launches
        h->launches += 1;
        return 2 * pairs;
    }
}

template <typename real, typename S>
int do_step(lbm_t *h, int n)
{
    const Params<real> P = make_params<real>(h);
    for (int it = 0; it < n; ++it) {
        {   // as many steps as possible before the next sampling step go into one cooperative launch (small lattices only)
            long run = n - it;
            if (h->mevery > 0) {
                const long k0 = h->step + 1;
                long ks = k0 <= h->mstart ? h->mstart : h->mstart + ((k0 - h->mstart + h->mevery - 1) / h->mevery) * h->mevery;
                run = std::min(run, ks - k0); // steps k0 .. ks-1 do not sample
            }
            const int done = run >= 4 ? try_step_loop<real, S>(h, P, (int)std::min(run, 1000000L)) : 0;
            if (done < 0) return done;
            if (done > 0) { h->step += done; it += done - 1; continue; }
        }
        const long k = h->step + 1;
        const bool sample = h->mevery > 0 && k >= h->mstart && (k - h->mstart) % h->mevery == 0;
        int rc = launch_step<real, S>(h, P, sample);
        if (rc) return rc;
        h->cur ^= 1;
        h->step = k;
        if (sample) h->mcount += 1;
    }
    return LBM_OK;
}

// box == nullptr: the whole lattice
inline Box whole_or(const lbm_t *h, const Box *box)
{
    if (box) return *box;
    Box b{};
    b.bn[0] = h->nx; b.bn[1] = h->ny; b.bn[2] = h->nz;
    return b;
}

template <typename real, typename S, typename out_t>
int do_get_macros(lbm_t *h, out_t *rho, out_t *ux, out_t *uy, out_t *uz, const Box *box = nullptr)
{
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_macros: flags not set");
    const Params<real> P = make_params<real>(h);
    const Box bx = whole_or(h, box);
    const long long NB = (long long)bx.bn[0] * bx.bn[1] * bx.bn[2];
    OutBuf o[4];
    out_t *dst[4] = {rho, ux, uy, uz};
    int rc = LBM_OK;
    int staged = 0;
    for (; staged < 4 && !rc; ++staged) rc = stage_out(h, dst[staged], (size_t)NB * sizeof(out_t), &o[staged]);
    if (!rc) {
        const int B = 256;
        if (h->inplace)
            macros_kernel<real, S, out_t, 1><<<blocks_for(NB, B), B, 0, h->stream>>>(
                (const S *)h->state(), h->flags(), (out_t *)o[0].dev, (out_t *)o[1].dev, (out_t *)o[2].dev, (out_t *)o[3].dev, P,
                (const real *)h->th_state(), h->links(), bx);
        else
            macros_kernel<real, S, out_t, 0><<<blocks_for(NB, B), B, 0, h->stream>>>(
                (const S *)h->state(), h->flags(), (out_t *)o[0].dev, (out_t *)o[1].dev, (out_t *)o[2].dev, (out_t *)o[3].dev, P,
                (const real *)h->th_state(), h->links(), bx);
        rc = check_launch(h, "macros_kernel");
    }
    int rc2 = finish_out(h, o, staged);
    return rc ? rc : rc2;
}

template <typename real, typename S, typename out_t>
int do_get_mean(lbm_t *h, out_t *ux, out_t *uy, out_t *uz, long *n_samples, const Box *box = nullptr)
{
    if (!h->want_mean) return fail(h, LBM_ESTATE, "get_mean: handle created without mean sums");
    const Params<real> P = make_params<real>(h);
    const Box bx = whole_or(h, box);
    const long long NB = (long long)bx.bn[0] * bx.bn[1] * bx.bn[2];
    if (n_samples) *n_samples = h->mcount;
    OutBuf o[3];
    out_t *dst[3] = {ux, uy, uz};
    int rc = LBM_OK;
    int staged = 0;
    for (; staged < 3 && !rc; ++staged) rc = stage_out(h, dst[staged], (size_t)NB * sizeof(out_t), &o[staged]);
    if (!rc) {
        const int B = 256;
        const double inv = h->mcount > 0 ? 1.0 / (double)h->mcount : 0.0;
        mean_out_kernel<real, out_t><<<blocks_for(NB, B), B, 0, h->stream>>>(
            (const real *)h->mean(), (out_t *)o[0].dev, (out_t *)o[1].dev, (out_t *)o[2].dev, inv, P, bx);
        rc = check_launch(h, "mean_out_kernel");
    }
    int rc2 = finish_out(h, o, staged);
    return rc ? rc : rc2;
}

template <typename real, typename S>
int do_get_links(lbm_t *h, uint32_t *links)
{
    const Params<real> P = make_params<real>(h);
    OutBuf o;
    int rc = stage_out(h, links, (size_t)P.N * sizeof(uint32_t), &o);
    if (rc) return rc;
    const int B = 256;
    links_out_kernel<real><<<blocks_for(P.N, B), B, 0, h->stream>>>(h->links(), h->flags(), (uint32_t *)o.dev, P);
    rc = check_launch(h, "links_out_kernel");
    int rc2 = finish_out(h, &o, 1);
    return rc ? rc : rc2;
}

template <typename real, typename S>
int do_get_state(lbm_t *h, double *f, const Box *box)
{
    const Params<real> P = make_params<real>(h);
    const Box bx = whole_or(h, box);
    const long long NB = (long long)bx.bn[0] * bx.bn[1] * bx.bn[2];
    OutBuf o;
    int rc = stage_out(h, f, (size_t)Q * NB * sizeof(double), &o);
    if (rc) return rc;
    const int B = 256;
    state_out_kernel<real, S><<<blocks_for(NB, B), B, 0, h->stream>>>((const S *)h->state(), h->flags(), h->links(), (double *)o.dev, P, bx);
    rc = check_launch(h, "state_out_kernel");
    int rc2 = finish_out(h, &o, 1);
    return rc ? rc : rc2;
}

// the whole lattice goes into buffer A, which becomes the current one (the first step rewrites every slot of B that is ever
// read); a box goes into the CURRENT buffer, whichever it is, and leaves the rest of the state alone
template <typename real, typename S>
int do_set_state(lbm_t *h, const double *f, const Box *box)
{
    const Params<real> P = make_params<real>(h);
    const Box bx = whole_or(h, box);
    const long long NB = (long long)bx.bn[0] * bx.bn[1] * bx.bn[2];
    InBuf in;
    int rc = stage_in(h, f, (size_t)Q * NB * sizeof(double), h->L.scratch_bytes, &in);
    if (rc) return rc;
    const int B = 256;
    S *dst = (S *)(box ? h->state() : h->bufA());
    state_in_kernel<real, S><<<blocks_for(NB, B), B, 0, h->stream>>>(dst, (S *)nullptr, (real *)h->fu(), h->flags(), h->links(),
                                                                   (const double *)in.dev, P, bx);
    rc = check_launch(h, "state_in_kernel");
    release_in(h, &in, 1);
    if (!rc && !h->inplace && !box) h->cur = 0;
    return rc;
}

template <typename real, typename S>
int do_balance_flux(lbm_t *h, double *before, double *after)
{
    const Params<real> P = make_params<real>(h);
    double *acc = (double *)h->scratch(); // acc[0..1] before, acc[2..3] after
    double host[4] = {0, 0, 0, 0};
    CUDA_TRY(h, cudaMemsetAsync(acc, 0, 4 * sizeof(double), h->stream));
    if (P.F > 0) {
        const int B = 128;
        const unsigned grid = blocks_for(P.F, B);
        flux_sum_kernel<real><<<grid, B, 0, h->stream>>>((const real *)h->fu(), h->flags(), acc, P);
        int rc = check_launch(h, "flux_sum_kernel");
        if (rc) return rc;
        flux_apply_kernel<real, S><<<grid, B, 0, h->stream>>>((S *)h->bufA(), (S *)h->bufB(), (real *)h->fu(), h->flags(), acc, P);
        rc = check_launch(h, "flux_apply_kernel");
        if (rc) return rc;
        flux_sum_kernel<real><<<grid, B, 0, h->stream>>>((const real *)h->fu(), h->flags(), acc + 2, P);
        rc = check_launch(h, "flux_sum_kernel");
        if (rc) return rc;
    }
    { int rc = thermal_refresh<real>(h); if (rc) return rc; }
    CUDA_TRY(h, cudaMemcpyAsync(host, acc, sizeof host, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (before) *before = host[0];
    if (after) *after = host[2];
    return LBM_OK;
}

template <typename real, typename S>
int do_refeed(lbm_t *h)
{
    const Params<real> P = make_params<real>(h);
    if (P.F == 0) return LBM_OK;
    const int B = 256;
    refeed_kernel<real, S><<<blocks_for(P.N, B), B, 0, h->stream>>>((const S *)h->state(), (real *)h->fu(), h->flags(), h->links(), P,
                                                                  (const real *)h->th_state());
    return check_launch(h, "refeed_kernel");
}

template <typename real, typename S>
int do_feed(lbm_t *dst, const lbm_t *src, int sx)
{
    const Params<real> D = make_params<real>(dst), Ps = make_params<real>(src);
    const int B = 128;
    const bool cross = src->stream != dst->stream;
    cudaEvent_t ev = nullptr;
    if (cross) {
        // the plane is read on dst's stream: order it after everything queued on src's stream (the precursor's last step) ...
        CUDA_TRY(dst, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        cudaError_t e = cudaEventRecord(ev, src->stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(dst->stream, ev, 0);
        if (e != cudaSuccess) { cudaEventDestroy(ev); return fail(dst, LBM_ECUDA, std::string("feed_inlet: ") + cudaGetErrorString(e)); }
    }
    feed_kernel<real, S><<<blocks_for((long long)D.ny * D.nz, B), B, 0, dst->stream>>>(
        (S *)dst->bufA(), (S *)dst->bufB(), (real *)dst->fu(), dst->flags(), D, (const S *)src->state(), src->flags(), src->links(), Ps, sx);
    int rc = check_launch(dst, "feed_kernel");
    if (cross) {
        // ... and what src does next after the read: its step after next rewrites the buffer this plane lies in, and src's
        // stream may run ahead of dst's by any number of steps
        cudaError_t e = cudaEventRecord(ev, dst->stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(src->stream, ev, 0);
        cudaEventDestroy(ev); // released once the recorded work has completed
        if (e != cudaSuccess && !rc) rc = fail(dst, LBM_ECUDA, std::string("feed_inlet: ") + cudaGetErrorString(e));
    }
    return rc ? rc : thermal_refresh<real>(dst);
}

} // namespace

// ---- C ABI -------------------------------------------------------------------------------------------------------------

template <typename real, typename S, typename in_t>
int do_set_theta(lbm_t *h, const in_t *theta, const in_t *ux, const in_t *uy, const in_t *uz)
{
    const Params<real> P = make_params<real>(h);
    const size_t bytes = (size_t)P.N * sizeof(in_t);
    InBuf in[4] = {};
    const in_t *src[4] = {theta, ux, uy, uz};
    int rc = LBM_OK;
    for (int k = 0; k < 4 && !rc; ++k) rc = stage_in(h, src[k], bytes, h->L.scratch_bytes, &in[k]);
    if (!rc) {
        const int B = 256;
        real *H0 = (real *)h->th_ws, *H1 = (real *)(h->th_ws + h->th_half());
        thermal_init_kernel<real, in_t><<<blocks_for(P.N, B), B, 0, h->stream>>>(
            H0, H1, h->flags(), h->links(), (const in_t *)in[0].dev, (const in_t *)in[1].dev, (const in_t *)in[2].dev,
            (const in_t *)in[3].dev, P, (const real *)h->state(), (real *)h->fu(), (real *)h->ft());
        rc = check_launch(h, "thermal_init_kernel");
    }
    release_in(h, in, 4);
    return rc;
}

template <typename in_t>
int set_theta_any(lbm_t *h, const in_t *theta, const in_t *ux, const in_t *uy, const in_t *uz)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->thermal) return fail(h, LBM_ESTATE, "set_theta: thermal lattice is off (lbm_set_thermal)");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "set_theta: flags not set");
    return DISPATCH_T(h, do_set_theta, in_t, h, theta, ux, uy, uz);
}

template <typename real, typename S, typename out_t>
int do_get_theta(lbm_t *h, out_t *theta)
{
    const Params<real> P = make_params<real>(h);
    OutBuf o[1];
    int rc = stage_out(h, theta, (size_t)P.N * sizeof(out_t), &o[0]);
    if (!rc) {
        const int B = 256;
        theta_out_kernel<real, out_t><<<blocks_for(P.N, B), B, 0, h->stream>>>((const real *)h->th_state(), h->flags(), (out_t *)o[0].dev, P);
        rc = check_launch(h, "theta_out_kernel");
    }
    int rc2 = finish_out(h, o, 1);
    return rc ? rc : rc2;
}

template <typename out_t>
int get_theta_any(lbm_t *h, out_t *theta)
{
    if (!h || !theta) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->thermal) return fail(h, LBM_ESTATE, "get_theta: thermal lattice is off (lbm_set_thermal)");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_theta: flags not set");
    return DISPATCH_T(h, do_get_theta, out_t, h, theta);
}

template <typename real>
int do_thermal_state(lbm_t *h, double *out, const double *in)
{
    const Params<real> P = make_params<real>(h);
    const size_t bytes = (size_t)QT * P.N * sizeof(double);
    const int B = 256;
    if (out) {
        OutBuf o;
        int rc = stage_out(h, out, bytes, &o);
        if (rc) return rc;
        thermal_state_out_kernel<real><<<blocks_for(P.N, B), B, 0, h->stream>>>((const real *)h->th_state(), h->flags(), (double *)o.dev, P);
        rc = check_launch(h, "thermal_state_out_kernel");
        int rc2 = finish_out(h, &o, 1);
        return rc ? rc : rc2;
    }
    InBuf ib;
    int rc = stage_in(h, in, bytes, h->L.scratch_bytes, &ib);
    if (rc) return rc;
    real *H0 = (real *)h->th_ws, *H1 = (real *)(h->th_ws + h->th_half());
    thermal_state_in_kernel<real><<<blocks_for(P.N, B), B, 0, h->stream>>>(H0, H1, h->flags(), h->links(), (const double *)ib.dev, P,
                                                                           (const real *)h->state(), (real *)h->fu(), (real *)h->ft());
    rc = check_launch(h, "thermal_state_in_kernel");
    release_in(h, &ib, 1);
    return rc;
}

namespace {
// theta_b[nz] -> the EQ_FIXED slots and cells (thermal_inlet_kernel); theta_b == nullptr refreshes the cells from the slots
template <typename real, typename in_t>
int do_inlet_theta(lbm_t *h, const in_t *theta_b)
{
    const Params<real> P = make_params<real>(h);
    if (P.F == 0) return LBM_OK;
    InBuf in;
    int rc = stage_in(h, theta_b, (size_t)h->nz * sizeof(in_t), 0, &in);
    if (rc) return rc;
    const int B = 128;
    real *H0 = (real *)h->th_ws, *H1 = (real *)(h->th_ws + h->th_half());
    thermal_inlet_kernel<real, in_t><<<blocks_for(P.F, B), B, 0, h->stream>>>(H0, H1, h->flags(), (const in_t *)in.dev, (const real *)h->fu(),
                                                                              (real *)h->ft(), P);
    rc = check_launch(h, "thermal_inlet_kernel");
    release_in(h, &in, 1);
    return rc;
}
} // namespace
template <typename in_t>
int set_inlet_theta_any(lbm_t *h, const in_t *theta_b)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!theta_b) return fail(h, LBM_EINVAL, "set_inlet_theta: NULL");
    if (!h->thermal) return fail(h, LBM_ESTATE, "set_inlet_theta: thermal lattice is off (lbm_set_thermal)");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "set_inlet_theta: flags not set");
    int rc = h->fp64 ? do_inlet_theta<double, in_t>(h, theta_b) : do_inlet_theta<float, in_t>(h, theta_b);
    // inflow fluctuations on: the side array holds u_b(step + 1); the cells belong to u_b(step) (reading 28)
    if (!rc && h->nmodes > 0) rc = DISPATCH(h, turb_publish, h, true);
    return rc;
}

bool has_eq_face(const int face[6])
{
    for (int k = 0; k < 6; ++k)
        if (face[k] == FACE_EQ_FIXED || face[k] == FACE_EQ_OUTFLOW) return true;
    return false;
}

extern "C" {

int lbm_set_thermal(lbm_t *h, double alpha, double g_beta, double theta_ref)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!(alpha > 0.0) || !std::isfinite(alpha) || !std::isfinite(g_beta) || !std::isfinite(theta_ref))
        return fail(h, LBM_EINVAL, "set_thermal: alpha must be > 0 and all arguments finite");
    if (h->s16) return fail(h, LBM_EINVAL, "set_thermal: not combinable with 16-bit population storage");
    if (!h->th_ws) CUDA_TRY(h, cudaMalloc((void **)&h->th_ws, 2 * h->th_half() + h->ft_bytes()));
    CUDA_TRY(h, cudaMemsetAsync(h->th_ws, 0, 2 * h->th_half() + h->ft_bytes(), h->stream)); // theta_ref at rest (shifted storage), theta_b = theta_ref
    h->alpha = alpha; h->gbeta = g_beta; h->theta_ref = theta_ref; h->thermal = true;
    int rc = LBM_OK;
    // open faces (reading 27): the EQ_FIXED cells hold h_eq(theta_ref, u_b) until lbm_set_inlet_theta says otherwise
    if (h->have_flags && has_eq_face(h->face)) rc = h->fp64 ? do_inlet_theta<double, float>(h, nullptr) : do_inlet_theta<float, float>(h, nullptr);
    // inflow fluctuations on: the cells hold u_b(step), the side array u_b(step + 1) — rewrite both lattices' cells for the velocity they have now (reading 28)
    if (!rc && h->have_flags && h->nmodes > 0) rc = DISPATCH(h, turb_publish, h, true);
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return rc;
}
int lbm_set_inlet_theta(lbm_t *h, const float *theta_b) { return set_inlet_theta_any<float>(h, theta_b); }
int lbm_set_inlet_theta_f64(lbm_t *h, const double *theta_b) { return set_inlet_theta_any<double>(h, theta_b); }
int lbm_set_theta(lbm_t *h, const float *theta, const float *ux, const float *uy, const float *uz) { return set_theta_any<float>(h, theta, ux, uy, uz); }
int lbm_set_theta_f64(lbm_t *h, const double *theta, const double *ux, const double *uy, const double *uz) { return set_theta_any<double>(h, theta, ux, uy, uz); }
int lbm_set_thermal_walls(lbm_t *h, const int on[6], const double theta_w[6])
{
    if (!h) return LBM_EINVAL;
    if (!on || !theta_w) return fail(h, LBM_EINVAL, "set_thermal_walls: NULL");
    if (!h->thermal) return fail(h, LBM_ESTATE, "set_thermal_walls: thermal lattice is off (lbm_set_thermal)");
    int mask = 0;
    for (int k = 0; k < 6; ++k) {
        if (!on[k]) continue;
        if (h->face[k] != LBM_WALL) return fail(h, LBM_EINVAL, "set_thermal_walls: only WALL faces can be held at a temperature");
        if (!std::isfinite(theta_w[k])) return fail(h, LBM_EINVAL, "set_thermal_walls: temperature not finite");
        mask |= 1 << k;
    }
    h->thd = mask;
    for (int k = 0; k < 6; ++k) h->thw[k] = on[k] ? theta_w[k] : 0.0;
    return LBM_OK;
}
int lbm_get_thermal_state(lbm_t *h, double *hpop)
{
    if (!h || !hpop) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->thermal) return fail(h, LBM_ESTATE, "get_thermal_state: thermal lattice is off (lbm_set_thermal)");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_thermal_state: flags not set");
    return h->fp64 ? do_thermal_state<double>(h, hpop, nullptr) : do_thermal_state<float>(h, hpop, nullptr);
}
int lbm_set_thermal_state(lbm_t *h, const double *hpop)
{
    if (!h || !hpop) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->thermal) return fail(h, LBM_ESTATE, "set_thermal_state: thermal lattice is off (lbm_set_thermal)");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "set_thermal_state: flags not set");
    return h->fp64 ? do_thermal_state<double>(h, nullptr, hpop) : do_thermal_state<float>(h, nullptr, hpop);
}
int lbm_get_theta(lbm_t *h, float *theta) { return get_theta_any<float>(h, theta); }
int lbm_get_theta_f64(lbm_t *h, double *theta) { return get_theta_any<double>(h, theta); }

int lbm_workspace_bytes(int nx, int ny, int nz, int want_mean, int precision, size_t *out)
{
    if (!out || !size_ok(nx, ny, nz)) return LBM_EINVAL;
    const int inplace = (precision >= 0 && (precision & LBM_STREAM_INPLACE)) ? 1 : 0;
    if (precision >= 0) precision &= ~LBM_STREAM_INPLACE;
    if (precision != LBM_PREC_F32 && precision != LBM_PREC_F64 && precision != LBM_PREC_F32_S16) return LBM_EINVAL;
    *out = make_layout(nx, ny, nz, want_mean, precision, inplace).total;
    return LBM_OK;
}

int lbm_create_ex(int nx, int ny, int nz, double nu0, double Cs, double f_cor, const double F[3], void *dev_workspace,
                  size_t workspace_bytes, void *cuda_stream, int precision, int want_mean, lbm_t **out)
{
    if (!out) return LBM_EINVAL;
    *out = nullptr;
    if (!size_ok(nx, ny, nz)) return LBM_EINVAL;
    const int inplace = (precision >= 0 && (precision & LBM_STREAM_INPLACE)) ? 1 : 0;
    if (precision >= 0) precision &= ~LBM_STREAM_INPLACE;
    if (precision != LBM_PREC_F32 && precision != LBM_PREC_F64 && precision != LBM_PREC_F32_S16) return LBM_EINVAL;
    if (!(nu0 > 0.0) || Cs < 0.0 || !std::isfinite(nu0) || !std::isfinite(Cs) || !std::isfinite(f_cor)) return LBM_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return LBM_ECUDA; }
    lbm_t *h = new (std::nothrow) lbm();
    if (!h) return LBM_ENOMEM;
    h->nx = nx; h->ny = ny; h->nz = nz;
    h->nu0 = nu0; h->Cs = Cs; h->fv[0] = 0.0; h->fv[1] = 0.0; h->fv[2] = f_cor;
    for (int a = 0; a < 3; ++a) h->F[a] = F ? F[a] : 0.0;
    const int def[6] = {LBM_EQ_FIXED, LBM_EQ_OUTFLOW, LBM_PERIODIC, LBM_PERIODIC, LBM_WALL, LBM_FREE_SLIP};
    for (int k = 0; k < 6; ++k) h->face[k] = def[k];
    h->precision = precision; h->fp64 = precision == LBM_PREC_F64; h->s16 = precision == LBM_PREC_F32_S16;
    h->want_mean = want_mean ? 1 : 0;
    h->inplace = inplace;
    h->L = make_layout(nx, ny, nz, h->want_mean, precision, inplace);
    h->stream = (cudaStream_t)cuda_stream;
    if (cudaGetDevice(&h->device) != cudaSuccess) { cudaGetLastError(); delete h; return LBM_ECUDA; }
    h->cur = 0; h->have_flags = false; h->step = 0;
    h->mstart = 0; h->mevery = 0; h->mcount = 0; h->launches = 0; h->variant = 0; h->damp_on = false; h->nmodes = 0; h->loop_ok = 0;
    h->thermal = false; h->alpha = 0; h->gbeta = 0; h->theta_ref = 0; h->th_ws = nullptr; h->thd = 0;
    for (int k = 0; k < 6; ++k) h->thw[k] = 0.0;
    for (int a = 0; a < 3; ++a) { h->dlo[a] = 0; h->dhi[a] = 0; }
    for (int k = 0; k < 4; ++k) h->slots[k] = lbm::Slot{nullptr, 0, false};
    if (dev_workspace) {
        if (workspace_bytes < h->L.total || ((uintptr_t)dev_workspace % ALIGN) != 0 || !is_device_ptr(dev_workspace)) {
            delete h;
            return LBM_EINVAL;
        }
        h->ws = (char *)dev_workspace; h->own_ws = false;
    } else {
        void *p = nullptr;
        cudaError_t e = cudaMalloc(&p, h->L.total);
        if (e != cudaSuccess) { cudaGetLastError(); delete h; return e == cudaErrorMemoryAllocation ? LBM_ENOMEM : LBM_ECUDA; }
        h->ws = (char *)p; h->own_ws = true;
    }
    *out = h;
    return LBM_OK;
}

int lbm_create(int nx, int ny, int nz, double nu0, double Cs, double f_cor, const double F[3], lbm_t **out)
{
    return lbm_create_ex(nx, ny, nz, nu0, Cs, f_cor, F, nullptr, 0, nullptr, 0, 1, out);
}

int lbm_destroy(lbm_t *h)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    cudaStreamSynchronize(h->stream);
    if (h->own_ws) cudaFree(h->ws);
    if (h->th_ws) cudaFree(h->th_ws);
    for (int k = 0; k < 4; ++k)
        if (h->slots[k].p) cudaFree(h->slots[k].p);
    delete h;
    return LBM_OK;
}

int lbm_set_boundaries(lbm_t *h, const int face_type[6])
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!face_type) return fail(h, LBM_EINVAL, "set_boundaries: NULL");
    for (int a = 0; a < 3; ++a) {
        const int lo = face_type[2 * a], hi = face_type[2 * a + 1];
        if (lo < 0 || lo > 4 || hi < 0 || hi > 4) return fail(h, LBM_EINVAL, "set_boundaries: unknown face type");
        if ((lo == LBM_PERIODIC) != (hi == LBM_PERIODIC)) return fail(h, LBM_EINVAL, "set_boundaries: PERIODIC must be set on both faces of an axis");
    }
    for (int k = 0; k < 6; ++k) h->face[k] = face_type[k];
    for (int k = 0; k < 6; ++k)
        if (face_type[k] != LBM_WALL) h->thd &= ~(1 << k); // a face that stops being a WALL is no longer held at a temperature
    h->have_flags = false;
    return LBM_OK;
}

int lbm_set_coriolis(lbm_t *h, const double f[3])
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!f) return fail(h, LBM_EINVAL, "set_coriolis: NULL");
    for (int a = 0; a < 3; ++a)
        if (!std::isfinite(f[a])) return fail(h, LBM_EINVAL, "set_coriolis: not finite");
    for (int a = 0; a < 3; ++a) h->fv[a] = f[a];
    return LBM_OK;
}

int lbm_set_damping(lbm_t *h, const int width[6], const double peak[6], const double *target)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!width || !peak) return fail(h, LBM_EINVAL, "set_damping: NULL");
    bool any = false;
    for (int k = 0; k < 6; ++k) {
        if (width[k] < 0 || !(peak[k] >= 0.0) || peak[k] > 1.0) return fail(h, LBM_EINVAL, "set_damping: need width >= 0 and 0 <= peak <= 1");
        any |= width[k] > 0 && peak[k] > 0.0;
    }
    // the outflow cells' next velocities are local macros of the current state: re-evaluate them under the new zones
    auto refeed = [&]() { return !h->have_flags ? LBM_OK : (DISPATCH(h, do_refeed, h)); };
    if (!any) {
        const bool was = h->damp_on;
        h->damp_on = false;
        return was ? refeed() : LBM_OK;
    }
    if (!target) return fail(h, LBM_EINVAL, "set_damping: target is NULL");
    if (is_device_ptr(target)) return fail(h, LBM_EINVAL, "set_damping: target must be a host array");
    // per-axis tables in double, then cast to the handle's precision: ramp = peak sin^2((pi/2)(1 - d/width)), d = cells
    // from the face layer; an axis table holds the larger of its two faces' ramps
    const int n[3] = {h->nx, h->ny, h->nz};
    const size_t cnt = (size_t)h->nx + h->ny + 4 * (size_t)h->nz;
    std::vector<double> t(cnt, 0.0);
    size_t base = 0;
    for (int a = 0; a < 3; ++a) {
        for (int c = 0; c < n[a]; ++c) {
            double s = 0.0;
            for (int side = 0; side < 2; ++side) {
                const int k = 2 * a + side, d = side ? n[a] - 1 - c : c;
                if (width[k] <= 0 || d >= width[k]) continue;
                const double r = std::sin(1.5707963267948966 * (1.0 - (double)d / (double)width[k]));
                s = std::max(s, peak[k] * r * r);
            }
            t[base + c] = s;
        }
        base += n[a];
    }
    for (size_t k = 0; k < 3 * (size_t)h->nz; ++k) {
        if (!std::isfinite(target[k])) return fail(h, LBM_EINVAL, "set_damping: target not finite");
        t[base + k] = target[k];
    }
    cudaError_t e;
    if (h->fp64) e = cudaMemcpyAsync(h->damp(), t.data(), cnt * sizeof(double), cudaMemcpyHostToDevice, h->stream);
    else {
        std::vector<float> tf(t.begin(), t.end());
        e = cudaMemcpyAsync(h->damp(), tf.data(), cnt * sizeof(float), cudaMemcpyHostToDevice, h->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream); // tf dies at the end of this block
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(h, LBM_ECUDA, std::string("set_damping: ") + cudaGetErrorString(e));
    for (int a = 0; a < 3; ++a) {
        const bool lo_on = width[2 * a] > 0 && peak[2 * a] > 0.0, hi_on = width[2 * a + 1] > 0 && peak[2 * a + 1] > 0.0;
        h->dlo[a] = lo_on ? std::min(width[2 * a], n[a]) : 0;
        h->dhi[a] = hi_on ? std::max(n[a] - width[2 * a + 1], 0) : n[a];
    }
    h->damp_on = true;
    return refeed();
}

int lbm_set_inflow_turbulence(lbm_t *h, int n_modes, const double *modes, double u_rms, double k_e, double k_eta)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->have_flags) return fail(h, LBM_ESTATE, "set_inflow_turbulence: flags not set");
    if (n_modes < 0 || n_modes > MAX_MODES) return fail(h, LBM_EINVAL, "set_inflow_turbulence: n_modes out of range");
    auto rewrite = [&]() { return DISPATCH(h, turb_publish, h, true); };
    if (n_modes == 0) {
        if (h->nmodes == 0) return LBM_OK;
        h->nmodes = 0;
        int rc = rewrite(); // no modes: the cells and the side array return to the mean
        if (!rc) CUDA_TRY(h, cudaStreamSynchronize(h->stream));
        return rc;
    }
    if (!modes || is_device_ptr(modes)) return fail(h, LBM_EINVAL, "set_inflow_turbulence: modes must be a host array");
    if (!(k_e > 0.0) || !(u_rms >= 0.0) || !(k_eta >= 0.0) || !std::isfinite(k_e) || !std::isfinite(u_rms) || !std::isfinite(k_eta))
        return fail(h, LBM_EINVAL, "set_inflow_turbulence: need k_e > 0, u_rms >= 0, k_eta >= 0");
    // device table [n][8]: kappa, a = 2 uhat sigma, psi, omega;  uhat = sqrt(E(|kappa|) dkappa), E = von Karman-Pao
    std::vector<double> t((size_t)n_modes * 8);
    for (int n = 0; n < n_modes; ++n) {
        const double *m = modes + 9 * (size_t)n;
        for (int c = 0; c < 9; ++c)
            if (!std::isfinite(m[c])) return fail(h, LBM_EINVAL, "set_inflow_turbulence: table not finite");
        if (m[8] < 0.0) return fail(h, LBM_EINVAL, "set_inflow_turbulence: dkappa < 0");
        const double k = std::sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]), r = k / k_e;
        double E = 1.453 * (u_rms * u_rms / k_e) * (r * r) * (r * r) / std::pow(1.0 + r * r, 17.0 / 6.0);
        if (k_eta > 0.0) E *= std::exp(-2.0 * (k / k_eta) * (k / k_eta));
        const double amp = 2.0 * std::sqrt(E * m[8]);
        double *d = t.data() + 8 * (size_t)n;
        d[0] = m[0]; d[1] = m[1]; d[2] = m[2];
        d[3] = amp * m[3]; d[4] = amp * m[4]; d[5] = amp * m[5];
        d[6] = m[6]; d[7] = m[7];
    }
    const Layout &L = h->L;
    if (h->nmodes == 0) // switching on: what the EQ slots hold now is the mean (both halves agree for EQ_FIXED slots)
        CUDA_TRY(h, cudaMemcpyAsync(h->fum(), h->fu(), L.fu_bytes / 2, cudaMemcpyDeviceToDevice, h->stream));
    CUDA_TRY(h, cudaMemcpyAsync(h->modes(), t.data(), t.size() * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    h->nmodes = n_modes;
    int rc = rewrite();
    CUDA_TRY(h, cudaStreamSynchronize(h->stream)); // t (host staging) must outlive the copy
    return rc;
}

int lbm_set_flags_mask(lbm_t *h, const int32_t *height, const uint8_t *solid)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!solid) return lbm_set_flags(h, height);
    h->nmodes = 0;
    const uint8_t *dev = solid;
    if (!is_device_ptr(solid)) { // a host mask is parked in the link-word area (4 Np bytes, rewritten by classify afterwards)
        CUDA_TRY(h, cudaMemcpyAsync(h->links(), solid, (size_t)h->N(), cudaMemcpyHostToDevice, h->stream));
        dev = (const uint8_t *)h->links();
    }
    int rc = DISPATCH(h, do_set_flags, h, height, dev, 1);
    if (!rc && dev != solid) CUDA_TRY(h, cudaStreamSynchronize(h->stream)); // the caller's buffer is free on return
    return rc;
}

int lbm_set_flags_mesh(lbm_t *h, const int32_t *height, int n_tri, const float *tri, int min_votes)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (n_tri < 0 || (n_tri > 0 && !tri)) return fail(h, LBM_EINVAL, "set_flags_mesh: bad triangle array");
    if (min_votes < 1 || min_votes > 3) return fail(h, LBM_EINVAL, "set_flags_mesh: min_votes must be 1, 2 or 3");
    h->nmodes = 0;
    InBuf in;
    int rc = stage_in(h, tri, (size_t)n_tri * 9 * sizeof(float), 0, &in);
    if (rc) return rc;
    uint8_t *votes = nullptr;
    rc = mesh_votes(h, n_tri, (const float *)in.dev, &votes);
    release_in(h, &in, 1);
    if (rc) return rc;
    // the heightmap staging of do_set_flags may reuse the scratch area now: the triangles are consumed
    return DISPATCH(h, do_set_flags, h, height, votes, min_votes);
}

int lbm_set_flags(lbm_t *h, const int32_t *height)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    h->nmodes = 0; // a new voxelisation resets the state and the boundary velocities
    return DISPATCH(h, do_set_flags, h, height);
}

int lbm_set_inlet_profile(lbm_t *h, const float *u, const float *v, const float *w) { return set_inlet_profile_any<float>(h, u, v, w); }
int lbm_set_inlet_profile_f64(lbm_t *h, const double *u, const double *v, const double *w) { return set_inlet_profile_any<double>(h, u, v, w); }
int lbm_set_inlet_plane(lbm_t *h, int face, const float *uvw) { return set_inlet_plane_any<float>(h, face, uvw); }
int lbm_set_inlet_plane_f64(lbm_t *h, int face, const double *uvw) { return set_inlet_plane_any<double>(h, face, uvw); }

int lbm_feed_inlet(lbm_t *dst, const lbm_t *src, int src_x_plane)
{
    if (!dst || !src) return LBM_EINVAL;
    DevGuard dg_(dst);
    if (!dst->have_flags || !src->have_flags) return fail(dst, LBM_ESTATE, "feed_inlet: flags not set");
    if (dst->nmodes > 0) return fail(dst, LBM_ESTATE, "feed_inlet: the mean boundary state is fixed while inflow fluctuations are on");
    if (dst->precision != src->precision) return fail(dst, LBM_EINVAL, "feed_inlet: precision mismatch");
    if (dst->nz != src->nz) return fail(dst, LBM_EINVAL, "feed_inlet: nz mismatch");
    if (src_x_plane < 0 || src_x_plane >= src->nx) return fail(dst, LBM_EINVAL, "feed_inlet: plane out of range");
    return DISPATCH(dst, do_feed, dst, src, src_x_plane);
}

int lbm_balance_flux(lbm_t *h, double *flux_before, double *flux_after)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->have_flags) return fail(h, LBM_ESTATE, "balance_flux: flags not set");
    if (h->nmodes > 0) return fail(h, LBM_ESTATE, "balance_flux: the mean boundary state is fixed while inflow fluctuations are on");
    return DISPATCH(h, do_balance_flux, h, flux_before, flux_after);
}

int lbm_set_macros(lbm_t *h, const float *rho, const float *ux, const float *uy, const float *uz)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    return DISPATCH_T(h, do_set_macros, float, h, rho, ux, uy, uz);
}
int lbm_set_macros_f64(lbm_t *h, const double *rho, const double *ux, const double *uy, const double *uz)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    return DISPATCH_T(h, do_set_macros, double, h, rho, ux, uy, uz);
}

int lbm_step(lbm_t *h, int n)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (n < 0) return fail(h, LBM_EINVAL, "step: n < 0");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "step: flags not set");
    return DISPATCH(h, do_step, h, n);
}

int lbm_mean_config(lbm_t *h, long start_step, int every)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->want_mean) return fail(h, LBM_ESTATE, "mean_config: handle created without mean sums");
    if (every < 0 || start_step < 0) return fail(h, LBM_EINVAL, "mean_config: negative argument");
    h->mstart = start_step; h->mevery = every;
    return LBM_OK;
}

int lbm_mean_reset(lbm_t *h)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->want_mean) return fail(h, LBM_ESTATE, "mean_reset: handle created without mean sums");
    CUDA_TRY(h, cudaMemsetAsync(h->mean(), 0, (size_t)3 * h->L.stride * (h->fp64 ? 8 : 4), h->stream));
    h->mcount = 0;
    return LBM_OK;
}

int lbm_get_macros(lbm_t *h, float *rho, float *ux, float *uy, float *uz)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    return DISPATCH_T(h, do_get_macros, float, h, rho, ux, uy, uz);
}
int lbm_get_macros_f64(lbm_t *h, double *rho, double *ux, double *uy, double *uz)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    return DISPATCH_T(h, do_get_macros, double, h, rho, ux, uy, uz);
}

int lbm_get_mean(lbm_t *h, float *ux, float *uy, float *uz, long *n_samples)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    return DISPATCH_T(h, do_get_mean, float, h, ux, uy, uz, n_samples);
}
int lbm_get_mean_f64(lbm_t *h, double *ux, double *uy, double *uz, long *n_samples)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    return DISPATCH_T(h, do_get_mean, double, h, ux, uy, uz, n_samples);
}

int lbm_get_flags(lbm_t *h, uint8_t *flags)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!flags) return fail(h, LBM_EINVAL, "get_flags: NULL");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_flags: flags not set");
    OutBuf o;
    int rc = stage_out(h, flags, (size_t)h->N(), &o);
    if (rc) return rc;
    const int B = 256;
    const Params<float> P = make_params<float>(h);
    flags_out_kernel<float><<<blocks_for(h->N(), B), B, 0, h->stream>>>(h->flags(), (uint8_t *)o.dev, P);
    rc = check_launch(h, "flags_out_kernel");
    int rc2 = finish_out(h, &o, 1);
    return rc ? rc : rc2;
}

int lbm_get_links(lbm_t *h, uint32_t *links)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!links) return fail(h, LBM_EINVAL, "get_links: NULL");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_links: flags not set");
    return DISPATCH(h, do_get_links, h, links);
}

int lbm_get_state(lbm_t *h, double *f)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!f) return fail(h, LBM_EINVAL, "get_state: NULL");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_state: flags not set");
    return DISPATCH(h, do_get_state, h, f, nullptr);
}

int lbm_set_state(lbm_t *h, const double *f)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!f) return fail(h, LBM_EINVAL, "set_state: NULL");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "set_state: flags not set");
    int rc = DISPATCH(h, do_set_state, h, f, nullptr);
    // the state brought its own boundary cells; the next launch must still find u_b(step + 1) in the side array
    if (!rc && h->nmodes > 0) rc = DISPATCH(h, turb_publish, h, false);
    return rc;
}

static int check_box(lbm_t *h, const int lo[3], const int hi[3], Box *bx, const char *what)
{
    if (!lo || !hi) return fail(h, LBM_EINVAL, std::string(what) + ": NULL");
    const int n[3] = {h->nx, h->ny, h->nz};
    for (int a = 0; a < 3; ++a) {
        if (lo[a] < 0 || hi[a] > n[a] || lo[a] >= hi[a]) return fail(h, LBM_EINVAL, std::string(what) + ": need 0 <= lo < hi <= n on every axis");
        bx->lo[a] = lo[a]; bx->bn[a] = hi[a] - lo[a];
    }
    return LBM_OK;
}

int lbm_get_state_box(lbm_t *h, const int lo[3], const int hi[3], double *f)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!f) return fail(h, LBM_EINVAL, "get_state_box: NULL");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_state_box: flags not set");
    Box bx{};
    int rc = check_box(h, lo, hi, &bx, "get_state_box");
    if (rc) return rc;
    return DISPATCH(h, do_get_state, h, f, &bx);
}

int lbm_set_state_box(lbm_t *h, const int lo[3], const int hi[3], const double *f)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!f) return fail(h, LBM_EINVAL, "set_state_box: NULL");
    if (!h->have_flags) return fail(h, LBM_ESTATE, "set_state_box: flags not set");
    Box bx{};
    int rc = check_box(h, lo, hi, &bx, "set_state_box");
    if (rc) return rc;
    rc = DISPATCH(h, do_set_state, h, f, &bx);
    if (!rc && h->nmodes > 0) rc = DISPATCH(h, turb_publish, h, false);
    return rc;
}

int lbm_get_macros_box(lbm_t *h, const int lo[3], const int hi[3], float *rho, float *ux, float *uy, float *uz)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_macros_box: flags not set");
    Box bx{};
    int rc = check_box(h, lo, hi, &bx, "get_macros_box");
    if (rc) return rc;
    return DISPATCH_T(h, do_get_macros, float, h, rho, ux, uy, uz, &bx);
}
int lbm_get_macros_box_f64(lbm_t *h, const int lo[3], const int hi[3], double *rho, double *ux, double *uy, double *uz)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_macros_box: flags not set");
    Box bx{};
    int rc = check_box(h, lo, hi, &bx, "get_macros_box");
    if (rc) return rc;
    return DISPATCH_T(h, do_get_macros, double, h, rho, ux, uy, uz, &bx);
}
int lbm_get_mean_box(lbm_t *h, const int lo[3], const int hi[3], float *ux, float *uy, float *uz, long *n_samples)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (!h->have_flags) return fail(h, LBM_ESTATE, "get_mean_box: flags not set");
    Box bx{};
    int rc = check_box(h, lo, hi, &bx, "get_mean_box");
    if (rc) return rc;
    return DISPATCH_T(h, do_get_mean, float, h, ux, uy, uz, n_samples, &bx);
}

long lbm_get_step(const lbm_t *h) { return h ? h->step : -1; }
int lbm_set_step(lbm_t *h, long step)
{
    if (!h || step < 0) return LBM_EINVAL;
    DevGuard dg_(h);
    h->step = step;
    if (h->nmodes > 0 && h->have_flags) return DISPATCH(h, turb_publish, h, false);
    return LBM_OK;
}

int lbm_sync(lbm_t *h)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

const char *lbm_last_error(const lbm_t *h) { return h ? h->err.c_str() : "NULL handle"; }
long lbm_launch_count(const lbm_t *h) { return h ? h->launches : -1; }

int lbm_lattice(int *c, int *opposite)
{
    if (!c || !opposite) return LBM_EINVAL;
    for (int i = 0; i < Q; ++i) {
        c[3 * i + 0] = dir_cx(i); c[3 * i + 1] = dir_cy(i); c[3 * i + 2] = dir_cz(i);
        opposite[i] = dir_opp(i);
    }
    return LBM_OK;
}

int lbm_set_variant(lbm_t *h, int variant)
{
    if (!h) return LBM_EINVAL;
    DevGuard dg_(h);
    if (variant < 0 || variant >= N_VARIANTS) return fail(h, LBM_EINVAL, "set_variant: unknown variant");
    h->variant = variant;
    return LBM_OK;
}

} // extern "C"

// ---- mesh voxeliser without a handle and without any allocation ---------------------------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
// The scratch of the ray-cast passes (one vote byte and one toggle byte per cell, one error word) lives in a file-scope
// device array of LBM_STATIC_VOXEL_MAX_CELLS cells: every GPU that loads this library holds its 4 MiB until exit.
// Every call shares the array and it keeps the last call's contents: the call clears what must start at zero, and two
// calls that overlap on the GPU (different streams, different host threads) RACE — serialise them.
namespace {

constexpr size_t SV_MAX_CELLS = LBM_STATIC_VOXEL_MAX_CELLS;
constexpr size_t SV_VOTES_OFF = 0;                               // votes   [SV_MAX_CELLS] bytes
constexpr size_t SV_TOG_OFF = SV_MAX_CELLS;                      // toggles [SV_MAX_CELLS + 256] bytes (words, padded)
constexpr size_t SV_ERR_OFF = 2 * SV_MAX_CELLS + 256;            // one int
constexpr size_t SV_BYTES = 2 * SV_MAX_CELLS + 512;
static_assert(SV_MAX_CELLS % 256 == 0, "offsets must stay 256-byte aligned");

static __device__ __align__(256) unsigned char g_static_voxel_scratch[SV_BYTES];

// In host code the array's name is a host-side stand-in, NOT a device address: the address a kernel may use comes from
// cudaGetSymbolAddress, asked once per device with that device current, and cached here.
constexpr int SV_MAX_DEVICES = 64;
unsigned char *g_sv_addr[SV_MAX_DEVICES] = {};

int static_voxel_scratch(unsigned char **out, char *err, size_t err_len)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess && (dev < 0 || dev >= SV_MAX_DEVICES)) {
        if (err && err_len) snprintf(err, err_len, "voxelise_mesh_static: device index %d beyond %d", dev, SV_MAX_DEVICES - 1);
        return LBM_EINVAL;
    }
    if (e == cudaSuccess && !g_sv_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_voxel_scratch);
        if (e == cudaSuccess) g_sv_addr[dev] = (unsigned char *)p;
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        if (err && err_len) snprintf(err, err_len, "voxelise_mesh_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
        return LBM_ECUDA;
    }
    *out = g_sv_addr[dev];
    return LBM_OK;
}

// solid[c] = votes[c] >= min_votes
__global__ void static_voxel_out_kernel(const uint8_t *__restrict__ votes, uint8_t *__restrict__ solid, long long N, int min_votes)
{
    const long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (c < N) solid[c] = votes[c] >= min_votes ? 1 : 0;
}

} // namespace

extern "C" int lbm_voxelise_mesh_static(int nx, int ny, int nz, int n_tri, const float *dev_tri, int min_votes, uint8_t *dev_solid,
                                        void *cuda_stream, char *err, size_t err_len)
{
    auto bad = [&](int code, const char *msg) {
        if (err && err_len) snprintf(err, err_len, "voxelise_mesh_static: %s", msg);
        return code;
    };
    if (err && err_len) err[0] = 0;
    if (nx < 1 || ny < 1 || nz < 1) return bad(LBM_EINVAL, "nx, ny, nz must be >= 1");
    const unsigned long long N = (unsigned long long)nx * (unsigned long long)ny * (unsigned long long)nz;
    if (N > SV_MAX_CELLS) {
        if (err && err_len)
            snprintf(err, err_len, "voxelise_mesh_static: %llu cells exceed the static scratch of %llu cells (LBM_STATIC_VOXEL_MAX_CELLS); "
                                   "use lbm_set_flags_mesh for larger boxes", N, (unsigned long long)SV_MAX_CELLS);
        return LBM_EINVAL;
    }
    if (n_tri < 0 || (n_tri > 0 && !dev_tri)) return bad(LBM_EINVAL, "bad triangle array");
    if (min_votes < 1 || min_votes > 3) return bad(LBM_EINVAL, "min_votes must be 1, 2 or 3");
    if (!dev_solid) return bad(LBM_EINVAL, "dev_solid is NULL");
    if (!is_device_ptr(dev_solid) || (n_tri > 0 && !is_device_ptr(dev_tri))) return bad(LBM_EINVAL, "tri and solid must be DEVICE pointers (nothing is staged: no allocation)");
    unsigned char *base = nullptr;
    int rc = static_voxel_scratch(&base, err, err_len);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint8_t *votes = base + SV_VOTES_OFF, *toggles = base + SV_TOG_OFF;
    int *errw = (int *)(base + SV_ERR_OFF);
    const size_t tog_bytes = align_up((size_t)N, 4) + 4;
    cudaError_t e = cudaMemsetAsync(votes, 0, (size_t)N, st);               // the array keeps the last call's contents
    if (e == cudaSuccess) e = cudaMemsetAsync(errw, 0, sizeof(int), st);
    const int B = 128;
    const unsigned tg = blocks_for((long long)n_tri * 32, B);
    const int n[3] = {nx, ny, nz};
    for (int d = 0; d < 3 && n_tri > 0 && e == cudaSuccess; ++d) {
        e = cudaMemsetAsync(toggles, 0, tog_bytes, st);
        if (e != cudaSuccess) break;
        const unsigned sg = blocks_for((long long)n[(d + 1) % 3] * n[(d + 2) % 3], B);
        if (d == 0) {
            mesh_toggle_kernel<0><<<tg, B, 0, st>>>(dev_tri, n_tri, (uint32_t *)toggles, nx, ny, nz, errw);
            mesh_scan_kernel<0><<<sg, B, 0, st>>>(toggles, votes, nx, ny, nz);
        } else if (d == 1) {
            mesh_toggle_kernel<1><<<tg, B, 0, st>>>(dev_tri, n_tri, (uint32_t *)toggles, nx, ny, nz, errw);
            mesh_scan_kernel<1><<<sg, B, 0, st>>>(toggles, votes, nx, ny, nz);
        } else {
            mesh_toggle_kernel<2><<<tg, B, 0, st>>>(dev_tri, n_tri, (uint32_t *)toggles, nx, ny, nz, errw);
            mesh_scan_kernel<2><<<sg, B, 0, st>>>(toggles, votes, nx, ny, nz);
        }
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        static_voxel_out_kernel<<<blocks_for((long long)N, 256), 256, 0, st>>>(votes, dev_solid, (long long)N, min_votes);
        e = cudaGetLastError();
    }
    int badv = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&badv, errw, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        cudaGetLastError();
        if (err && err_len) snprintf(err, err_len, "voxelise_mesh_static: %s", cudaGetErrorString(e));
        return LBM_ECUDA;
    }
    if (badv) return bad(LBM_EINVAL, "a vertex is not finite or outside [-1024, 2048) cells");
    return LBM_OK;
}
