// lb_b200.cu -- the C-ABI library of include/lb.h: context, transfers, and the general
// ("two-pass") kernels that work for any box shape.  The bandwidth-optimised one-pass step
// lives in lb_onepass.cuh.  sm_100a only; there is no CPU path in this file or anywhere in
// the library.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>

#include "../../include/lb.h"
#include "lb_lattice.cuh"
#include "lb_onepass.cuh"

using namespace lb;

// ----------------------------------------------------------------------------------------
// context
// ----------------------------------------------------------------------------------------
struct lb_ctx {
    int nx, ny, nz;
    long long N;       // nodes
    long long NP;      // plane stride in elements: N rounded up so every [k][i] plane is 256-B aligned
    int dtype;
    double tau[2], G;
    cudaStream_t stream;
    bool own_stream;
    void* f[2];        // ping-pong population buffers, [k][i][NP]
    int cur;           // f[cur] holds time t
    void* rho;         // [k][NP] densities (two-pass path and getters)
    unsigned int* links;   // N words: bit i = neighbour i solid, bit 31 = this node solid
    bool has_solid;
    bool have_fields;
    int kernel;        // resolved LB_KERNEL_*
    int kernel_req;
    double* stage;     // device staging, STAGE_NODES * 5 doubles
    double* diag_part; // [DIAG_BLOCKS][5]
    double* diag_out;  // [5]
    long long launches;
};

namespace {

constexpr long long STAGE_NODES = 1ll << 22;
constexpr int DIAG_BLOCKS = 148 * 8;
constexpr unsigned SOLID_BIT = 1u << 31;

thread_local std::string g_err;

int fail(int code, const char* what) { g_err = what; return code; }
int fail_cuda(cudaError_t e, const char* where) {
    g_err = std::string(where) + ": " + cudaGetErrorString(e);
    return LB_ECUDA;
}
#define CU(call)                                                         \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return fail_cuda(e__, #call);            \
    } while (0)

size_t esize(const lb_ctx* c) { return c->dtype == LB_F64 ? 8 : 4; }

template <typename T> __device__ __forceinline__ T* plane(T* f, long long NP, int k, int i) { return f + (long long)(k * Q + i) * NP; }
template <typename T> __device__ __forceinline__ const T* plane(const T* f, long long NP, int k, int i) { return f + (long long)(k * Q + i) * NP; }

// ----------------------------------------------------------------------------------------
// setup / transfer kernels (not on the hot path)
// ----------------------------------------------------------------------------------------
// f_i^k = feq_i(rho^k, u) for nodes [n0, n0+cnt); staged inputs are doubles (Eq. 10).
template <typename T>
__global__ void k_init_eq(T* __restrict__ f, long long NP, long long n0, long long cnt,
                          const double* __restrict__ s_rr, const double* __restrict__ s_rb,
                          const double* __restrict__ s_ux, const double* __restrict__ s_uy,
                          const double* __restrict__ s_uz, const unsigned* __restrict__ links) {
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= cnt) return;
    const long long n = n0 + t;
    const bool solid = links && (links[n] & SOLID_BIT);
    const T ux = s_ux ? T(s_ux[t]) : T(0), uy = s_uy ? T(s_uy[t]) : T(0), uz = s_uz ? T(s_uz[t]) : T(0);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        T fe[Q];
        equilibrium19<T>(fe, T(k == 0 ? s_rr[t] : s_rb[t]), ux, uy, uz);
#pragma unroll
        for (int i = 0; i < Q; ++i) plane(f, NP, k, i)[n] = solid ? T(0) : fe[i];
    }
}

template <typename T>
__global__ void k_zero_solids(T* __restrict__ f, long long NP, long long N, const unsigned* __restrict__ links) {
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= N || !(links[n] & SOLID_BIT)) return;
#pragma unroll
    for (int q = 0; q < NPOP; ++q) f[(long long)q * NP + n] = T(0);
}

// widen/narrow one [k][i] plane chunk between the context type and the ABI's double
template <typename T>
__global__ void k_to_double(const T* __restrict__ src, double* __restrict__ dst, long long cnt) {
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < cnt) dst[t] = double(src[t]);
}
template <typename T>
__global__ void k_from_double(const double* __restrict__ src, T* __restrict__ dst, long long cnt) {
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < cnt) dst[t] = T(src[t]);
}

// links[n]: bit i iff fluid n has a solid neighbour along c_i; bit 31 iff n itself is solid.
__global__ void k_build_links(const unsigned char* __restrict__ mask, unsigned* __restrict__ links,
                              int nx, int ny, int nz) {
    const long long N = (long long)nx * ny * nz;
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= N) return;
    const int x = int(n % nx), y = int((n / nx) % ny), z = int(n / ((long long)nx * ny));
    unsigned m = 0;
    if (mask[n]) {
        m = SOLID_BIT;
    } else {
#pragma unroll
        for (int i = 1; i < Q; ++i) {
            const int xn = (x + dir_cx(i) + nx) % nx, yn = (y + dir_cy(i) + ny) % ny, zn = (z + dir_cz(i) + nz) % nz;
            if (mask[xn + (long long)nx * (yn + (long long)ny * zn)]) m |= 1u << i;
        }
    }
    links[n] = m;
}

__global__ void k_links_out(const unsigned* __restrict__ links, unsigned* __restrict__ out, long long cnt) {
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < cnt) out[t] = links[t] & ~SOLID_BIT;
}

// rho^k, u for nodes [n0, n0+cnt) into double staging (Eq. 6-7); solids and empty nodes report 0.
template <typename T>
__global__ void k_moments_out(const T* __restrict__ f, long long NP, long long n0, long long cnt,
                              double* __restrict__ o_rr, double* __restrict__ o_rb, double* __restrict__ o_ux,
                              double* __restrict__ o_uy, double* __restrict__ o_uz) {
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= cnt) return;
    const long long n = n0 + t;
    T r[2], jx = T(0), jy = T(0), jz = T(0);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        T fk[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) fk[i] = plane(f, NP, k, i)[n];
        T ax, ay, az;
        moments19<T>(fk, r[k], ax, ay, az);
        jx += ax; jy += ay; jz += az;
    }
    const T rt = r[0] + r[1];
    const T inv = rt != T(0) ? T(1) / rt : T(0);
    o_rr[t] = double(r[0]); o_rb[t] = double(r[1]);
    o_ux[t] = double(jx * inv); o_uy[t] = double(jy * inv); o_uz[t] = double(jz * inv);
}

// ----------------------------------------------------------------------------------------
// diagnostics: warp shuffle -> block -> fixed-order final pass (deterministic)
// ----------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <typename T>
__global__ void __launch_bounds__(256) k_diag_partial(const T* __restrict__ f, long long NP, long long N,
                                                      double* __restrict__ part) {
    double acc[5] = {0, 0, 0, 0, 0};
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < N; n += (long long)gridDim.x * blockDim.x) {
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            T fk[Q];
#pragma unroll
            for (int i = 0; i < Q; ++i) fk[i] = plane(f, NP, k, i)[n];
            T r, ax, ay, az;
            moments19<T>(fk, r, ax, ay, az);
            acc[k] += double(r); acc[2] += double(ax); acc[3] += double(ay); acc[4] += double(az);
        }
    }
    __shared__ double sm[5][8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < 5; ++q) {
        const double s = warp_sum(acc[q]);
        if (lane == 0) sm[q][wid] = s;
    }
    __syncthreads();
    if (threadIdx.x < 5) {
        double s = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) s += sm[threadIdx.x][w];
        part[blockIdx.x * 5 + threadIdx.x] = s;
    }
}

__global__ void __launch_bounds__(256) k_diag_final(const double* __restrict__ part, int nblocks, double* __restrict__ out) {
    __shared__ double sm[256];
    for (int q = 0; q < 5; ++q) {
        double s = 0;
        for (int b = threadIdx.x; b < nblocks; b += 256) s += part[b * 5 + q];
        sm[threadIdx.x] = s;
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) {
            if (threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) out[q] = sm[0];
        __syncthreads();
    }
}

// ----------------------------------------------------------------------------------------
// two-pass time step, any box shape
// ----------------------------------------------------------------------------------------
// pass 1: rho^k = sum_i f_i^k (Eq. 6).  Solid nodes hold zero populations, so they report 0.
template <typename T>
__global__ void __launch_bounds__(256) k_density(const T* __restrict__ f, long long NP, long long N, T* __restrict__ rho) {
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= N) return;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        T r = plane(f, NP, k, 0)[n];
#pragma unroll
        for (int i = 1; i < Q; ++i) r += plane(f, NP, k, i)[n];
        rho[(long long)k * NP + n] = r;
    }
}

// pass 2: Shan-Chen force, BGK collision with forcing, bounce-back, periodic streaming (push).
template <typename T, bool HAS_SOLID>
__global__ void __launch_bounds__(256) k_collide_stream(const T* __restrict__ f, T* __restrict__ g,
                                                        const T* __restrict__ rho, const unsigned* __restrict__ links,
                                                        long long NP, int nx, int ny, int nz,
                                                        T om_r, T om_b, T G) {
    const long long N = (long long)nx * ny * nz;
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= N) return;
    unsigned lk = 0;
    if (HAS_SOLID) {
        lk = links[n];
        if (lk & SOLID_BIT) return;              // no computation inside a particle
    }
    const int x = int(n % nx), y = int((n / nx) % ny), z = int(n / ((long long)nx * ny));
    const int xs[3] = {x == 0 ? nx - 1 : x - 1, x, x == nx - 1 ? 0 : x + 1};
    const long long ys[3] = {(long long)nx * (y == 0 ? ny - 1 : y - 1), (long long)nx * y, (long long)nx * (y == ny - 1 ? 0 : y + 1)};
    const long long zs[3] = {(long long)nx * ny * (z == 0 ? nz - 1 : z - 1), (long long)nx * ny * z, (long long)nx * ny * (z == nz - 1 ? 0 : z + 1)};
    long long nb[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) nb[i] = xs[dir_cx(i) + 1] + ys[dir_cy(i) + 1] + zs[dir_cz(i) + 1];

    T fr[Q], fb[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) { fr[i] = plane(f, NP, 0, i)[n]; fb[i] = plane(f, NP, 1, i)[n]; }
    T rr, rb, jrx, jry, jrz, jbx, jby, jbz;
    moments19<T>(fr, rr, jrx, jry, jrz);
    moments19<T>(fb, rb, jbx, jby, jbz);
    // the densities this step's force was specified with are pass 1's (index-order sums)
    rr = rho[n]; rb = rho[NP + n];
    const T den = om_r * rr + om_b * rb;                            // S4
    const T inv = den != T(0) ? T(1) / den : T(0);
    const T ux = (om_r * jrx + om_b * jbx) * inv, uy = (om_r * jry + om_b * jby) * inv, uz = (om_r * jrz + om_b * jbz) * inv;
    // du^k = -G sum_i w_i rho^kbar(x+c_i) c_i  (S2, S3, S6); solids hold rho = 0 (S7)
    T gr[3] = {T(0), T(0), T(0)}, gb[3] = {T(0), T(0), T(0)};      // gradients of rho_b (acts on red) and rho_r (on blue)
#pragma unroll
    for (int p = 0; p < 9; ++p) {
        const T db = w_pair<T>(p) * (rho[NP + nb[2 * p + 1]] - rho[NP + nb[2 * p + 2]]);
        const T dr = w_pair<T>(p) * (rho[nb[2 * p + 1]] - rho[nb[2 * p + 2]]);
        if (pair_cx(p)) { gr[0] += T(pair_cx(p)) * db; gb[0] += T(pair_cx(p)) * dr; }
        if (pair_cy(p)) { gr[1] += T(pair_cy(p)) * db; gb[1] += T(pair_cy(p)) * dr; }
        if (pair_cz(p)) { gr[2] += T(pair_cz(p)) * db; gb[2] += T(pair_cz(p)) * dr; }
    }
    collide19<T>(fr, rr, T(1) - om_r, ux, uy, uz, ux - G * gr[0], uy - G * gr[1], uz - G * gr[2]);
    collide19<T>(fb, rb, T(1) - om_b, ux, uy, uz, ux - G * gb[0], uy - G * gb[1], uz - G * gb[2]);
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        if (HAS_SOLID && (lk >> i & 1u)) {                          // Eq. 23-24 with u_b = 0
            plane(g, NP, 0, dir_opp(i))[n] = fr[i];
            plane(g, NP, 1, dir_opp(i))[n] = fb[i];
        } else {                                                    // Eq. 5: streaming, periodic
            plane(g, NP, 0, i)[nb[i]] = fr[i];
            plane(g, NP, 1, i)[nb[i]] = fb[i];
        }
    }
}

inline unsigned blocks_for(long long cnt, int bs) { return unsigned((cnt + bs - 1) / bs); }

template <typename T>
int step_twopass(lb_ctx* c) {
    const T* f = static_cast<const T*>(c->f[c->cur]);
    T* g = static_cast<T*>(c->f[c->cur ^ 1]);
    T* rho = static_cast<T*>(c->rho);
    const unsigned nb = blocks_for(c->N, 256);
    k_density<T><<<nb, 256, 0, c->stream>>>(f, c->NP, c->N, rho);
    const T om_r = T(1.0 / c->tau[0]), om_b = T(1.0 / c->tau[1]), G = T(c->G);
    if (c->has_solid)
        k_collide_stream<T, true><<<nb, 256, 0, c->stream>>>(f, g, rho, c->links, c->NP, c->nx, c->ny, c->nz, om_r, om_b, G);
    else
        k_collide_stream<T, false><<<nb, 256, 0, c->stream>>>(f, g, rho, nullptr, c->NP, c->nx, c->ny, c->nz, om_r, om_b, G);
    c->launches += 2;
    CU(cudaGetLastError());
    c->cur ^= 1;
    return LB_OK;
}

template <typename T>
int zero_solids_both(lb_ctx* c) {
    for (int b = 0; b < 2; ++b) {
        k_zero_solids<T><<<blocks_for(c->N, 256), 256, 0, c->stream>>>(static_cast<T*>(c->f[b]), c->NP, c->N, c->links);
        c->launches++;
    }
    CU(cudaGetLastError());
    return LB_OK;
}

// ----------------------------------------------------------------------------------------
// one-pass time step (lb_onepass.cuh): boxes whose x, y sides are multiples of the 32 x 8 tile
// ----------------------------------------------------------------------------------------
constexpr int OP_TX = 32, OP_TY = 8;
constexpr int OP_RESIDENT_CTAS = 148 * 2;

bool onepass_ok(const lb_ctx* c) { return c->nx % OP_TX == 0 && c->ny % OP_TY == 0; }

// planes per CTA: long enough to amortise the 2-plane density prologue, short enough that the
// grid is many waves of the resident CTAs; a divisor of nz when one is close.
int onepass_zc(const lb_ctx* c) {
    if (const char* e = std::getenv("LB_ONEPASS_ZC")) { const int v = std::atoi(e); if (v >= 1) return v < c->nz ? v : c->nz; }
    const long long tiles = (long long)(c->nx / OP_TX) * (c->ny / OP_TY);
    const long long chunks_wanted = (OP_RESIDENT_CTAS * 6 + tiles - 1) / tiles;
    long long zc = c->nz / (chunks_wanted > 0 ? chunks_wanted : 1);
    if (zc > 64) zc = 64;
    if (zc < 16) zc = 16;
    if (zc > c->nz) zc = c->nz;
    for (long long d = zc; d >= (zc + 1) / 2; --d)
        if (c->nz % d == 0) return int(d);
    return int(zc);
}

template <typename T>
int step_onepass(lb_ctx* c) {
    const T* f = static_cast<const T*>(c->f[c->cur]);
    T* g = static_cast<T*>(c->f[c->cur ^ 1]);
    const int zc = onepass_zc(c);
    const dim3 grid(c->nx / OP_TX, c->ny / OP_TY, (c->nz + zc - 1) / zc);
    const T om_r = T(1.0 / c->tau[0]), om_b = T(1.0 / c->tau[1]), G = T(c->G);
    if (c->has_solid)
        k_step_onepass<T, true, OP_TX, OP_TY><<<grid, OP_TX * OP_TY, 0, c->stream>>>(f, g, c->links, c->NP, c->nx, c->ny, c->nz, zc, om_r, om_b, G);
    else
        k_step_onepass<T, false, OP_TX, OP_TY><<<grid, OP_TX * OP_TY, 0, c->stream>>>(f, g, nullptr, c->NP, c->nx, c->ny, c->nz, zc, om_r, om_b, G);
    c->launches += 1;
    CU(cudaGetLastError());
    c->cur ^= 1;
    return LB_OK;
}

int resolve_kernel(lb_ctx* c, int kind) {
    if (kind == LB_KERNEL_AUTO) return onepass_ok(c) ? LB_KERNEL_ONEPASS : LB_KERNEL_TWOPASS;
    if (kind == LB_KERNEL_ONEPASS && !onepass_ok(c)) return -1;
    return kind;
}

}  // namespace

// ----------------------------------------------------------------------------------------
// C ABI
// ----------------------------------------------------------------------------------------
extern "C" {

const char* lb_last_error(void) { return g_err.c_str(); }
const char* lb_version(void) { return "lb-b200 0.1 (sm_100a)"; }

lb_ctx* lb_create_ex(int nx, int ny, int nz, double tau_r, double tau_b, double G, int dtype, void* cuda_stream) {
    g_err.clear();
    if (nx < 1 || ny < 1 || nz < 1) { fail(LB_EINVAL, "box dimensions must be >= 1"); return nullptr; }
    if ((long long)nx * ny * nz > (1ll << 31) - 1) { fail(LB_EINVAL, "box too large (N must fit in 31 bits)"); return nullptr; }
    if (!(tau_r > 0.5) || !(tau_b > 0.5) || !std::isfinite(tau_r) || !std::isfinite(tau_b)) {
        fail(LB_EINVAL, "tau must be finite and > 0.5 (0 < omega < 2)"); return nullptr;
    }
    if (!std::isfinite(G)) { fail(LB_EINVAL, "G must be finite"); return nullptr; }
    if (dtype != LB_F64 && dtype != LB_F32) { fail(LB_EINVAL, "dtype must be LB_F64 or LB_F32"); return nullptr; }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        fail_cuda(e != cudaSuccess ? e : cudaErrorNoDevice, "no CUDA device (this library has no CPU fallback)");
        return nullptr;
    }
    lb_ctx* c = new (std::nothrow) lb_ctx();
    if (!c) { fail(LB_ENOMEM, "host allocation failed"); return nullptr; }
    std::memset(c, 0, sizeof(*c));
    c->nx = nx; c->ny = ny; c->nz = nz;
    c->N = (long long)nx * ny * nz;
    c->NP = (c->N + 63) / 64 * 64;
    c->dtype = dtype;
    c->tau[0] = tau_r; c->tau[1] = tau_b; c->G = G;
    if (cuda_stream) { c->stream = static_cast<cudaStream_t>(cuda_stream); c->own_stream = false; }
    else {
        e = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) { fail_cuda(e, "cudaStreamCreate"); delete c; return nullptr; }
        c->own_stream = true;
    }
    const size_t es = esize(c);
    const size_t fbytes = size_t(NPOP) * c->NP * es;
    bool ok = true;
    ok = ok && cudaMalloc(&c->f[0], fbytes) == cudaSuccess;
    ok = ok && cudaMalloc(&c->f[1], fbytes) == cudaSuccess;
    ok = ok && cudaMalloc(&c->rho, size_t(2) * c->NP * es) == cudaSuccess;
    ok = ok && cudaMalloc(&c->links, size_t(c->N) * sizeof(unsigned)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->stage, size_t(STAGE_NODES) * 5 * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->diag_part, size_t(DIAG_BLOCKS) * 5 * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->diag_out, 5 * sizeof(double)) == cudaSuccess;
    if (ok) {
        ok = ok && cudaMemsetAsync(c->f[0], 0, fbytes, c->stream) == cudaSuccess;
        ok = ok && cudaMemsetAsync(c->f[1], 0, fbytes, c->stream) == cudaSuccess;
        ok = ok && cudaMemsetAsync(c->rho, 0, size_t(2) * c->NP * es, c->stream) == cudaSuccess;
        ok = ok && cudaMemsetAsync(c->links, 0, size_t(c->N) * sizeof(unsigned), c->stream) == cudaSuccess;
    }
    if (!ok) {
        e = cudaGetLastError();
        g_err = std::string("device allocation failed: ") + cudaGetErrorString(e);
        lb_destroy(c);
        return nullptr;                                  // LB_ENOMEM
    }
    c->kernel_req = LB_KERNEL_AUTO;
    c->kernel = resolve_kernel(c, LB_KERNEL_AUTO);
    return c;
}

lb_ctx* lb_create(int nx, int ny, int nz, double tau_r, double tau_b, double G) {
    return lb_create_ex(nx, ny, nz, tau_r, tau_b, G, LB_F64, nullptr);
}

void lb_destroy(lb_ctx* c) {
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    cudaFree(c->f[0]); cudaFree(c->f[1]); cudaFree(c->rho); cudaFree(c->links);
    cudaFree(c->stage); cudaFree(c->diag_part); cudaFree(c->diag_out);
    if (c->own_stream) cudaStreamDestroy(c->stream);
    delete c;
}

int lb_sync(lb_ctx* c) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    CU(cudaStreamSynchronize(c->stream));
    return LB_OK;
}

long long lb_launch_count(const lb_ctx* c) { return c ? c->launches : 0; }

int lb_set_kernel(lb_ctx* c, int kind) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    if (kind != LB_KERNEL_AUTO && kind != LB_KERNEL_TWOPASS && kind != LB_KERNEL_ONEPASS) return fail(LB_EINVAL, "unknown kernel kind");
    const int r = resolve_kernel(c, kind);
    if (r < 0) return fail(LB_EINVAL, "box shape does not allow the one-pass kernel");
    c->kernel_req = kind;
    c->kernel = r;
    return LB_OK;
}

int lb_set_solid_mask(lb_ctx* c, const unsigned char* mask) {
    if (!c || !mask) return fail(LB_EINVAL, "NULL argument");
    unsigned char* d_mask = nullptr;
    CU(cudaMalloc(&d_mask, size_t(c->N)));
    cudaError_t e = cudaMemcpyAsync(d_mask, mask, size_t(c->N), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) {
        k_build_links<<<blocks_for(c->N, 256), 256, 0, c->stream>>>(d_mask, c->links, c->nx, c->ny, c->nz);
        c->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(d_mask);
    if (e != cudaSuccess) return fail_cuda(e, "lb_set_solid_mask");
    c->has_solid = true;   // a mask of all zeros still takes the (slower) link-checking kernels
    return c->dtype == LB_F64 ? zero_solids_both<double>(c) : zero_solids_both<float>(c);
}

int lb_set_fields(lb_ctx* c, const double* rho_r, const double* rho_b, const double* ux, const double* uy, const double* uz) {
    if (!c || !rho_r || !rho_b) return fail(LB_EINVAL, "NULL argument");
    const int nu = (ux != nullptr) + (uy != nullptr) + (uz != nullptr);
    if (nu != 0 && nu != 3) return fail(LB_EINVAL, "ux, uy, uz must be all NULL or all non-NULL");
    const double* src[5] = {rho_r, rho_b, ux, uy, uz};
    for (long long n0 = 0; n0 < c->N; n0 += STAGE_NODES) {
        const long long cnt = (c->N - n0 < STAGE_NODES) ? c->N - n0 : STAGE_NODES;
        double* st[5];
        for (int a = 0; a < 5; ++a) {
            st[a] = src[a] ? c->stage + a * STAGE_NODES : nullptr;
            if (src[a]) CU(cudaMemcpyAsync(st[a], src[a] + n0, size_t(cnt) * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        }
        const unsigned* lk = c->has_solid ? c->links : nullptr;
        if (c->dtype == LB_F64)
            k_init_eq<double><<<blocks_for(cnt, 128), 128, 0, c->stream>>>(static_cast<double*>(c->f[c->cur]), c->NP, n0, cnt, st[0], st[1], st[2], st[3], st[4], lk);
        else
            k_init_eq<float><<<blocks_for(cnt, 128), 128, 0, c->stream>>>(static_cast<float*>(c->f[c->cur]), c->NP, n0, cnt, st[0], st[1], st[2], st[3], st[4], lk);
        c->launches++;
        CU(cudaGetLastError());
    }
    CU(cudaStreamSynchronize(c->stream));          // the caller's arrays are free again
    c->have_fields = true;
    return LB_OK;
}

int lb_set_populations(lb_ctx* c, const double* f) {
    if (!c || !f) return fail(LB_EINVAL, "NULL argument");
    for (int q = 0; q < NPOP; ++q) {
        const double* src = f + (long long)q * c->N;
        if (c->dtype == LB_F64) {
            CU(cudaMemcpyAsync(static_cast<double*>(c->f[c->cur]) + (long long)q * c->NP, src, size_t(c->N) * 8, cudaMemcpyHostToDevice, c->stream));
        } else {
            float* dst = static_cast<float*>(c->f[c->cur]) + (long long)q * c->NP;
            for (long long n0 = 0; n0 < c->N; n0 += STAGE_NODES * 5) {
                const long long cnt = (c->N - n0 < STAGE_NODES * 5) ? c->N - n0 : STAGE_NODES * 5;
                CU(cudaMemcpyAsync(c->stage, src + n0, size_t(cnt) * 8, cudaMemcpyHostToDevice, c->stream));
                k_from_double<float><<<blocks_for(cnt, 256), 256, 0, c->stream>>>(c->stage, dst + n0, cnt);
                c->launches++;
                CU(cudaGetLastError());
            }
        }
    }
    if (c->has_solid) {
        const int rc = c->dtype == LB_F64 ? zero_solids_both<double>(c) : zero_solids_both<float>(c);
        if (rc != LB_OK) return rc;
    }
    CU(cudaStreamSynchronize(c->stream));
    c->have_fields = true;
    return LB_OK;
}

int lb_step(lb_ctx* c, int nsteps) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    if (nsteps < 0) return fail(LB_EINVAL, "nsteps must be >= 0");
    if (!c->have_fields) return fail(LB_ESTATE, "lb_step before lb_set_fields / lb_set_populations");
    for (int s = 0; s < nsteps; ++s) {
        int rc;
        if (c->kernel == LB_KERNEL_ONEPASS) rc = c->dtype == LB_F64 ? step_onepass<double>(c) : step_onepass<float>(c);
        else rc = c->dtype == LB_F64 ? step_twopass<double>(c) : step_twopass<float>(c);
        if (rc != LB_OK) return rc;
    }
    return LB_OK;
}

int lb_get_populations(lb_ctx* c, double* f) {
    if (!c || !f) return fail(LB_EINVAL, "NULL argument");
    for (int q = 0; q < NPOP; ++q) {
        double* dst = f + (long long)q * c->N;
        if (c->dtype == LB_F64) {
            CU(cudaMemcpyAsync(dst, static_cast<const double*>(c->f[c->cur]) + (long long)q * c->NP, size_t(c->N) * 8, cudaMemcpyDeviceToHost, c->stream));
        } else {
            const float* src = static_cast<const float*>(c->f[c->cur]) + (long long)q * c->NP;
            for (long long n0 = 0; n0 < c->N; n0 += STAGE_NODES * 5) {
                const long long cnt = (c->N - n0 < STAGE_NODES * 5) ? c->N - n0 : STAGE_NODES * 5;
                k_to_double<float><<<blocks_for(cnt, 256), 256, 0, c->stream>>>(src + n0, c->stage, cnt);
                c->launches++;
                CU(cudaGetLastError());
                CU(cudaMemcpyAsync(dst + n0, c->stage, size_t(cnt) * 8, cudaMemcpyDeviceToHost, c->stream));
            }
        }
    }
    CU(cudaStreamSynchronize(c->stream));
    return LB_OK;
}

int lb_get_moments(lb_ctx* c, double* rho_r, double* rho_b, double* ux, double* uy, double* uz) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    double* dst[5] = {rho_r, rho_b, ux, uy, uz};
    for (long long n0 = 0; n0 < c->N; n0 += STAGE_NODES) {
        const long long cnt = (c->N - n0 < STAGE_NODES) ? c->N - n0 : STAGE_NODES;
        double* st[5];
        for (int a = 0; a < 5; ++a) st[a] = c->stage + a * STAGE_NODES;
        if (c->dtype == LB_F64)
            k_moments_out<double><<<blocks_for(cnt, 128), 128, 0, c->stream>>>(static_cast<const double*>(c->f[c->cur]), c->NP, n0, cnt, st[0], st[1], st[2], st[3], st[4]);
        else
            k_moments_out<float><<<blocks_for(cnt, 128), 128, 0, c->stream>>>(static_cast<const float*>(c->f[c->cur]), c->NP, n0, cnt, st[0], st[1], st[2], st[3], st[4]);
        c->launches++;
        CU(cudaGetLastError());
        for (int a = 0; a < 5; ++a)
            if (dst[a]) CU(cudaMemcpyAsync(dst[a] + n0, st[a], size_t(cnt) * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    return LB_OK;
}

int lb_get_link_mask(lb_ctx* c, unsigned int* links) {
    if (!c || !links) return fail(LB_EINVAL, "NULL argument");
    unsigned* st = reinterpret_cast<unsigned*>(c->stage);
    const long long chunk = STAGE_NODES * 10;          // staging holds 5*STAGE_NODES doubles
    for (long long n0 = 0; n0 < c->N; n0 += chunk) {
        const long long cnt = (c->N - n0 < chunk) ? c->N - n0 : chunk;
        k_links_out<<<blocks_for(cnt, 256), 256, 0, c->stream>>>(c->links + n0, st, cnt);
        c->launches++;
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(links + n0, st, size_t(cnt) * sizeof(unsigned), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    return LB_OK;
}

int lb_get_diagnostics(lb_ctx* c, double mass[2], double momentum[3]) {
    if (!c || !mass || !momentum) return fail(LB_EINVAL, "NULL argument");
    if (c->dtype == LB_F64)
        k_diag_partial<double><<<DIAG_BLOCKS, 256, 0, c->stream>>>(static_cast<const double*>(c->f[c->cur]), c->NP, c->N, c->diag_part);
    else
        k_diag_partial<float><<<DIAG_BLOCKS, 256, 0, c->stream>>>(static_cast<const float*>(c->f[c->cur]), c->NP, c->N, c->diag_part);
    k_diag_final<<<1, 256, 0, c->stream>>>(c->diag_part, DIAG_BLOCKS, c->diag_out);
    c->launches += 2;
    CU(cudaGetLastError());
    double h[5];
    CU(cudaMemcpyAsync(h, c->diag_out, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    mass[0] = h[0]; mass[1] = h[1];
    momentum[0] = h[2]; momentum[1] = h[3]; momentum[2] = h[4];
    return LB_OK;
}

}  // extern "C"
