// lb_single.cu -- single-fluid D3Q19 BGK, fused collide + stream (the paper's "case 1", Table 1):
// the 304 B/node (fp64) / 152 B/node (fp32) calibration workload of SURVEY 8(f) N4, behind the lbs_* calls of include/lb.h.
//
// One component, no force: f_i(x + c_i, t + 1) = (1 - om) f_i(x, t) + om feq_i(rho, u)  (Eq. 1; Eq. 10,
// PAPER.md:338-342), periodic box.  Same state convention as the two-component library: the buffer holds the
// post-collision, not yet streamed values h_i(x); the reader streams (f_i(x) = h_i(x - c_i), "pull"), so stores are aligned
// and coalesced and only the loads of the 10 directions with c_x != 0 are shifted by one element.  Two buffers (the paper's
// "one-step two-grid").  One thread per node, a thread block = 128 consecutive x of one (y, z) row: no integer
// division, the y / z wrap is block-uniform.  Nothing is staged: every population is read once and written once, and the 19
// loads of a thread are independent (memory-level parallelism comes from occupancy).
#include <cuda_runtime.h>

#include <cmath>
#include <cstring>
#include <new>
#include <string>

#include "../../include/lb.h"
#include "lb_lattice.cuh"

using namespace lb;

struct lbs_ctx {
    int nx, ny, nz, dtype, device;
    long long N, NP;
    double tau;
    cudaStream_t stream;
    bool own_stream, have_fields;
    void* f[2];
    int cur;
    double* stage;          // 4 * stage_nodes doubles
    long long stage_nodes;
    long long launches;
};

void lb_set_error(int code, const char* what);          // lb_b200.cu: the library's one error slot per thread

namespace {

constexpr int BX = 128;
constexpr long long STAGE_NODES = 1ll << 22;

int sfail(int code, const char* what) { lb_set_error(code, what); return code; }
int sfail_cuda(cudaError_t e, const char* where) {
    const std::string m = std::string(where) + ": " + cudaGetErrorString(e);
    const int code = e == cudaErrorMemoryAllocation ? LB_ENOMEM : LB_ECUDA;
    lb_set_error(code, m.c_str());
    return code;
}
#define SCU(call)                                                        \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return sfail_cuda(e__, #call);           \
    } while (0)

struct Guard {
    int prev = -1;
    explicit Guard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) cudaSetDevice(dev); else prev = -1;
    }
    ~Guard() { if (prev >= 0) cudaSetDevice(prev); }
};

// node of this thread and the periodic offsets of its neighbours (block-uniform in y and z)
struct Where {
    long long n; int xm, x, xp; long long row[3], pln[3];
    __device__ __forceinline__ long long at(int dx, int dy, int dz) const { return pln[dz + 1] + row[dy + 1] + (dx < 0 ? xm : (dx > 0 ? xp : x)); }
};
__device__ __forceinline__ bool where(Where& w, int nx, int ny, int nz) {
    const int x = blockIdx.x * BX + threadIdx.x, y = blockIdx.y, z = blockIdx.z;
    if (x >= nx) return false;
    const long long pl = (long long)nx * ny;
    w.x = x; w.xm = x == 0 ? nx - 1 : x - 1; w.xp = x == nx - 1 ? 0 : x + 1;
    w.row[0] = (long long)nx * (y == 0 ? ny - 1 : y - 1); w.row[1] = (long long)nx * y; w.row[2] = (long long)nx * (y == ny - 1 ? 0 : y + 1);
    w.pln[0] = pl * (z == 0 ? nz - 1 : z - 1); w.pln[1] = pl * z; w.pln[2] = pl * (z == nz - 1 ? 0 : z + 1);
    w.n = w.pln[1] + w.row[1] + x;
    return true;
}

// the hot kernel: pull, moments (Eq. 6-7), BGK collision (Eq. 1, Eq. 10), aligned stores.  om is a run-time value.
template <typename T>
__global__ void __launch_bounds__(BX) k_single_step(const T* __restrict__ h, T* __restrict__ g, long long NP, int nx, int ny, int nz, T om) {
    Where w;
    if (!where(w, nx, ny, nz)) return;
    T f[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) f[i] = __ldg(h + (long long)i * NP + w.at(-dir_cx(i), -dir_cy(i), -dir_cz(i)));
    T rho, jx, jy, jz;
    moments19<T>(f, rho, jx, jy, jz);
    const T inv = rho != T(0) ? T(1) / rho : T(0);
    const T ux = jx * inv, uy = jy * inv, uz = jz * inv;
    collide19<T>(f, rho, T(1) - om, ux, uy, uz, ux, uy, uz);      // no force: the shifted velocity is the velocity itself
#pragma unroll
    for (int i = 0; i < Q; ++i) g[(long long)i * NP + w.n] = f[i];
}

// f_i = feq_i(rho, u) (Eq. 10) written as h-state: h_i(y) = f_i(y + c_i)
template <typename T>
__global__ void __launch_bounds__(BX) k_single_init(T* __restrict__ h, long long NP, int nx, int ny, int nz,
                                                    const double* __restrict__ rho, const double* __restrict__ ux,
                                                    const double* __restrict__ uy, const double* __restrict__ uz) {
    Where w;
    if (!where(w, nx, ny, nz)) return;
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        const long long m = w.at(dir_cx(i), dir_cy(i), dir_cz(i));
        T fe[Q];
        equilibrium19<T>(fe, T(rho[m]), ux ? T(ux[m]) : T(0), uy ? T(uy[m]) : T(0), uz ? T(uz[m]) : T(0));
        h[(long long)i * NP + w.n] = fe[i];
    }
}

// h-state <-> f (streaming, Eq. 5), one direction plane at a time into / out of the double staging buffer
template <typename T>
__global__ void __launch_bounds__(BX) k_single_stream_out(const T* __restrict__ h, double* __restrict__ out, long long NP, int nx, int ny, int nz, int i) {
    Where w;
    if (!where(w, nx, ny, nz)) return;
    const int cx = i == 0 ? 0 : dir_cx(i), cy = dir_cy(i), cz = dir_cz(i);
    out[w.n] = double(h[(long long)i * NP + w.at(-cx, -cy, -cz)]);
}
template <typename T>
__global__ void __launch_bounds__(BX) k_single_unstream_in(const double* __restrict__ in, T* __restrict__ h, long long NP, int nx, int ny, int nz, int i) {
    Where w;
    if (!where(w, nx, ny, nz)) return;
    h[(long long)i * NP + w.n] = T(in[w.at(dir_cx(i), dir_cy(i), dir_cz(i))]);
}

template <typename T>
__global__ void __launch_bounds__(BX) k_single_moments(const T* __restrict__ h, long long NP, int nx, int ny, int nz,
                                                       double* __restrict__ o_r, double* __restrict__ o_x, double* __restrict__ o_y, double* __restrict__ o_z) {
    Where w;
    if (!where(w, nx, ny, nz)) return;
    T f[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) f[i] = h[(long long)i * NP + w.at(-dir_cx(i), -dir_cy(i), -dir_cz(i))];
    T rho, jx, jy, jz;
    moments19<T>(f, rho, jx, jy, jz);
    const T inv = rho != T(0) ? T(1) / rho : T(0);
    o_r[w.n] = double(rho); o_x[w.n] = double(jx * inv); o_y[w.n] = double(jy * inv); o_z[w.n] = double(jz * inv);
}

dim3 grid_of(const lbs_ctx* c) { return dim3(unsigned((c->nx + BX - 1) / BX), unsigned(c->ny), unsigned(c->nz)); }

}  // namespace

extern "C" {

lbs_ctx* lbs_create(int nx, int ny, int nz, double tau, int dtype, void* cuda_stream) {
    lb_set_error(LB_OK, "");
    if (nx < 1 || ny < 1 || nz < 1 || ny > 65535 || nz > 65535) { sfail(LB_EINVAL, "box dimensions must be >= 1 (ny, nz <= 65535)"); return nullptr; }
    if ((long long)nx * ny * nz > (1ll << 31) - 1) { sfail(LB_EINVAL, "box too large (N must fit in 31 bits)"); return nullptr; }
    if (!(tau > 0.5) || !std::isfinite(tau)) { sfail(LB_EINVAL, "tau must be finite and > 0.5 (0 < omega < 2)"); return nullptr; }
    if (dtype != LB_F64 && dtype != LB_F32) { sfail(LB_EINVAL, "dtype must be LB_F64 or LB_F32"); return nullptr; }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) { sfail_cuda(e != cudaSuccess ? e : cudaErrorNoDevice, "no CUDA device (this library has no CPU fallback)"); return nullptr; }
    lbs_ctx* c = new (std::nothrow) lbs_ctx();
    if (!c) { sfail(LB_ENOMEM, "host allocation failed"); return nullptr; }
    std::memset(c, 0, sizeof(*c));
    cudaGetDevice(&c->device);
    c->nx = nx; c->ny = ny; c->nz = nz; c->dtype = dtype; c->tau = tau;
    c->N = (long long)nx * ny * nz;
    c->NP = (c->N + 63) / 64 * 64;
    if (cuda_stream) { c->stream = static_cast<cudaStream_t>(cuda_stream); c->own_stream = false; }
    else {
        e = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) { sfail_cuda(e, "cudaStreamCreate"); delete c; return nullptr; }
        c->own_stream = true;
    }
    const size_t es = dtype == LB_F64 ? 8 : 4;
    c->stage_nodes = c->N < STAGE_NODES ? c->N : STAGE_NODES;
    bool ok = cudaMalloc(&c->f[0], size_t(Q) * c->NP * es) == cudaSuccess;
    ok = ok && cudaMalloc(&c->f[1], size_t(Q) * c->NP * es) == cudaSuccess;
    ok = ok && cudaMalloc(&c->stage, size_t(4) * c->N * sizeof(double)) == cudaSuccess;   // whole fields: the init kernel reads neighbours
    if (!ok) {
        e = cudaGetLastError();
        lbs_destroy(c);
        sfail_cuda(e, "device allocation failed");
        return nullptr;
    }
    return c;
}

void lbs_destroy(lbs_ctx* c) {
    if (!c) return;
    Guard guard(c->device);
    cudaStreamSynchronize(c->stream);
    cudaFree(c->f[0]); cudaFree(c->f[1]); cudaFree(c->stage);
    if (c->own_stream) cudaStreamDestroy(c->stream);
    delete c;
}

int lbs_set_fields(lbs_ctx* c, const double* rho, const double* ux, const double* uy, const double* uz) {
    if (!c || !rho) return sfail(LB_EINVAL, "NULL argument");
    const int nu = (ux != nullptr) + (uy != nullptr) + (uz != nullptr);
    if (nu != 0 && nu != 3) return sfail(LB_EINVAL, "ux, uy, uz must be all NULL or all non-NULL");
    Guard guard(c->device);
    const double* src[4] = {rho, ux, uy, uz};
    double* st[4];
    for (int a = 0; a < 4; ++a) {
        st[a] = src[a] ? c->stage + a * c->N : nullptr;
        if (src[a]) SCU(cudaMemcpyAsync(st[a], src[a], size_t(c->N) * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    }
    if (c->dtype == LB_F64) k_single_init<double><<<grid_of(c), BX, 0, c->stream>>>(static_cast<double*>(c->f[c->cur]), c->NP, c->nx, c->ny, c->nz, st[0], st[1], st[2], st[3]);
    else k_single_init<float><<<grid_of(c), BX, 0, c->stream>>>(static_cast<float*>(c->f[c->cur]), c->NP, c->nx, c->ny, c->nz, st[0], st[1], st[2], st[3]);
    c->launches++;
    SCU(cudaGetLastError());
    SCU(cudaStreamSynchronize(c->stream));
    c->have_fields = true;
    return LB_OK;
}

int lbs_set_populations(lbs_ctx* c, const double* f) {
    if (!c || !f) return sfail(LB_EINVAL, "NULL argument");
    Guard guard(c->device);
    for (int i = 0; i < Q; ++i) {
        SCU(cudaMemcpyAsync(c->stage, f + (long long)i * c->N, size_t(c->N) * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        if (c->dtype == LB_F64) k_single_unstream_in<double><<<grid_of(c), BX, 0, c->stream>>>(c->stage, static_cast<double*>(c->f[c->cur]), c->NP, c->nx, c->ny, c->nz, i);
        else k_single_unstream_in<float><<<grid_of(c), BX, 0, c->stream>>>(c->stage, static_cast<float*>(c->f[c->cur]), c->NP, c->nx, c->ny, c->nz, i);
        c->launches++;
        SCU(cudaGetLastError());
    }
    SCU(cudaStreamSynchronize(c->stream));
    c->have_fields = true;
    return LB_OK;
}

int lbs_step(lbs_ctx* c, int nsteps) {
    if (!c) return sfail(LB_EINVAL, "NULL context");
    if (nsteps < 0) return sfail(LB_EINVAL, "nsteps must be >= 0");
    if (!c->have_fields) return sfail(LB_ESTATE, "lbs_step before lbs_set_fields / lbs_set_populations");
    Guard guard(c->device);
    for (int s = 0; s < nsteps; ++s) {
        if (c->dtype == LB_F64)
            k_single_step<double><<<grid_of(c), BX, 0, c->stream>>>(static_cast<const double*>(c->f[c->cur]), static_cast<double*>(c->f[c->cur ^ 1]), c->NP, c->nx, c->ny, c->nz, 1.0 / c->tau);
        else
            k_single_step<float><<<grid_of(c), BX, 0, c->stream>>>(static_cast<const float*>(c->f[c->cur]), static_cast<float*>(c->f[c->cur ^ 1]), c->NP, c->nx, c->ny, c->nz, float(1.0 / c->tau));
        c->launches++;
        SCU(cudaGetLastError());
        c->cur ^= 1;
    }
    return LB_OK;
}

int lbs_get_populations(lbs_ctx* c, double* f) {
    if (!c || !f) return sfail(LB_EINVAL, "NULL argument");
    Guard guard(c->device);
    for (int i = 0; i < Q; ++i) {
        if (c->dtype == LB_F64) k_single_stream_out<double><<<grid_of(c), BX, 0, c->stream>>>(static_cast<const double*>(c->f[c->cur]), c->stage, c->NP, c->nx, c->ny, c->nz, i);
        else k_single_stream_out<float><<<grid_of(c), BX, 0, c->stream>>>(static_cast<const float*>(c->f[c->cur]), c->stage, c->NP, c->nx, c->ny, c->nz, i);
        c->launches++;
        SCU(cudaGetLastError());
        SCU(cudaMemcpyAsync(f + (long long)i * c->N, c->stage, size_t(c->N) * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    }
    SCU(cudaStreamSynchronize(c->stream));
    return LB_OK;
}

int lbs_get_moments(lbs_ctx* c, double* rho, double* ux, double* uy, double* uz) {
    if (!c) return sfail(LB_EINVAL, "NULL context");
    Guard guard(c->device);
    double* st[4];
    for (int a = 0; a < 4; ++a) st[a] = c->stage + a * c->N;
    if (c->dtype == LB_F64) k_single_moments<double><<<grid_of(c), BX, 0, c->stream>>>(static_cast<const double*>(c->f[c->cur]), c->NP, c->nx, c->ny, c->nz, st[0], st[1], st[2], st[3]);
    else k_single_moments<float><<<grid_of(c), BX, 0, c->stream>>>(static_cast<const float*>(c->f[c->cur]), c->NP, c->nx, c->ny, c->nz, st[0], st[1], st[2], st[3]);
    c->launches++;
    SCU(cudaGetLastError());
    double* dst[4] = {rho, ux, uy, uz};
    for (int a = 0; a < 4; ++a)
        if (dst[a]) SCU(cudaMemcpyAsync(dst[a], st[a], size_t(c->N) * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    SCU(cudaStreamSynchronize(c->stream));
    return LB_OK;
}

int lbs_sync(lbs_ctx* c) {
    if (!c) return sfail(LB_EINVAL, "NULL context");
    Guard guard(c->device);
    SCU(cudaStreamSynchronize(c->stream));
    return LB_OK;
}

long long lbs_launch_count(const lbs_ctx* c) { return c ? c->launches : 0; }

}  // extern "C"
