// lb_b200.cu -- the C-ABI library of include/lb.h: context, transfers, and the general
// ("two-pass") kernels that work for any box shape.  The bandwidth-optimised one-pass step
// lives in lb_onepass.cuh.  sm_100a only; there is no CPU path in this file or anywhere in
// the library.
//
// Device state ("h-state", see lb_onepass.cuh): the population buffer f[cur] holds the
// post-collision, not yet streamed values h of the previous step; every reader streams while it
// reads (pull).  The ABI speaks f (streamed populations at their nodes, Eq. 5): k_unstream /
// k_stream convert on the way in / out.  They are pure moves, so set -> get is bit-exact.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include "../../include/lb.h"
#include "lb_lattice.cuh"
#include "lb_onepass.cuh"
#include "lb_tma.cuh"
#include "lb_halo.cuh"
#include "lb_node.cuh"

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
    int device;        // CUDA device the context lives on (the current device at lb_create*)
    cudaStream_t stream;
    bool own_stream;
    void* f[2];        // ping-pong population buffers, [k][i][NP]; f[cur] = h-state, f[cur^1] = scratch
    int cur;
    // density of the CURRENT time level as the four single-writer arrays of lb_onepass.cuh, ping-pong.
    // rho_x / rho_y / rho_xy exist only when the box takes the one-pass tile.
    void* rho_in[2]; void* rho_x[2]; void* rho_y[2]; void* rho_xy[2];
    long long s_x, s_y, s_xy;   // component strides (elements) of the edge arrays
    // the halo kernel (lb_halo.cuh): own-gather edge rows / columns (shapes of rho_y / rho_x), ping-pong with the others,
    // and the x-halo copies of the populations, one per population buffer
    void* rho_er[2]; void* rho_ec[2];
    void* hx[2];
    long long hx_elems;         // 20 * nz * (nx / 32) * ny
    bool hx_valid;     // hx[cur] matches f[cur]
    int rcur;
    bool rho_valid;    // the density arrays [rcur] hold the density of the state in f[cur], in the format rho_fmt
    int rho_fmt;       // RHO_FULL (rho_in + edge pieces: two-pass, one-pass, TMA kernels) or RHO_EDGE (frame arrays only: halo kernel)
    unsigned int* links;   // N words: bit i = neighbour i solid, bit 31 = this node solid
    bool has_solid;
    bool have_fields;
    int kernel;        // resolved LB_KERNEL_*
    int kernel_req;
    int zc;            // planes per CTA of the one-pass kernel
    int zc_tma;        // ... of the TMA kernel
    CUtensorMap tmap_hx[2];   // [buffer] x-halo box TY x 1 x 1 x 2 over hx [plane][z][tile_x][y]
    // later operators, both on the general two-pass path
    int model;         // LB_MODEL_SHAN_CHEN or LB_MODEL_COLOUR_GRADIENT
    double sigma, beta;
    bool in_set_spheres;
    int nsph;          // spheres with prescribed velocities (moving-wall bounce-back, force / torque per sphere)
    double radius;
    double* sph;       // device: centres[nsph][3], vel[nsph][3], omega[nsph][3], F[nsph][3], T[nsph][3]
    int* pid;          // device: sphere of every solid node (-1 = none)
    int diag_mode;     // LB_OPT_DIAG: the halo kernel also leaves the mass / momentum sums of the new state behind
    bool diag_fresh;   // diag_cta holds the per-CTA partials of the state in f[cur]
    double* diag_cta;  // [diag_cta_cap][5]
    long long diag_cta_cap;
    long long diag_ncta;
    CUtensorMap tmap[2][3];   // [buffer][narrow box 32 x 8, wide box (32 + 16 B) x 8, wrapped-column box 16 B x 8; each 2 planes deep] over [plane][z][y][x]
    bool have_tmap;
    double* stage;     // device staging, stage_nodes * 5 doubles
    long long stage_nodes;   // min(N, STAGE_NODES)
    int zc_req;        // lb_set_option(LB_OPT_ZC): planes per CTA of the one-pass kernels, 0 = heuristic
    double* diag_part; // [DIAG_BLOCKS][5]
    double* diag_out;  // [5]
    bool balance;      // tma_grid: pad the CTA count to a multiple of the SM count (LB_OPT_BALANCE)
    double* na_scratch; // device address of g_noalloc_scratch on this context's device (lb_diagnostics_noalloc), nullptr if unknown
    long long launches;
};

namespace {

constexpr long long STAGE_NODES = 1ll << 22;
constexpr int DIAG_BLOCKS = 148 * 8;
constexpr unsigned SOLID_BIT = 1u << 31;
constexpr int OP_TX = 32, OP_TY = 8;
enum { RHO_FULL = 0, RHO_EDGE = 1 };

thread_local std::string g_err;
thread_local int g_err_code = LB_OK;

int fail(int code, const char* what) { g_err = what; g_err_code = code; return code; }
int fail_cuda(cudaError_t e, const char* where) {
    g_err = std::string(where) + ": " + cudaGetErrorString(e);
    g_err_code = e == cudaErrorMemoryAllocation ? LB_ENOMEM : LB_ECUDA;
    return g_err_code;
}

// ---- lb_diagnostics_noalloc: scratch that exists without any allocation call ----------------------------
// One partial (5 doubles) per block of k_diag_partial, each block taking NOALLOC_NODES_PER_BLOCK nodes: 16384 blocks x 40 B =
// 640 KB, held by every GPU that loads the library until the process exits; enough for 2^28 nodes (512^3 = 2^27).
// In host code `g_noalloc_scratch` is a host-side stand-in, NOT a device address: the address a kernel can use comes from
// cudaGetSymbolAddress, asked for once per device with that device current (noalloc_scratch_address, called by lb_create_ex).
constexpr int NOALLOC_MAX_BLOCKS = 16384;
constexpr long long NOALLOC_NODES_PER_BLOCK = 16384;       // 256 threads x 64 nodes
}  // namespace
static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_MAX_BLOCKS * 5];
namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
double* g_noalloc_addr[NOALLOC_MAX_DEVICES] = {};
// device address of the scratch array on `device`, which must be the current device; nullptr (error slot set) on failure
double* noalloc_scratch_address(int device) {
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) { fail(LB_EINVAL, "lb_diagnostics_noalloc: device ordinal beyond the address table"); return nullptr; }
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_addr[device]) {
        double* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_noalloc_scratch);
        if (e != cudaSuccess) { fail_cuda(e, "cudaGetSymbolAddress(g_noalloc_scratch)"); return nullptr; }
        g_noalloc_addr[device] = ptr;
    }
    return g_noalloc_addr[device];
}

// every ABI call runs on the context's device, whatever the caller's current device is
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) cudaSetDevice(dev); else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define CU(call)                                                         \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return fail_cuda(e__, #call);            \
    } while (0)

size_t esize(const lb_ctx* c) { return c->dtype == LB_F64 ? 8 : 4; }

template <typename T> __device__ __forceinline__ T* plane(T* f, long long NP, int k, int i) { return f + (long long)pop_plane(k, i) * NP; }
template <typename T> __device__ __forceinline__ const T* plane(const T* f, long long NP, int k, int i) { return f + (long long)pop_plane(k, i) * NP; }

// periodic neighbour offsets of node n, any box shape
struct Nbr {
    long long o[3][3];    // o[0][dx+1] x offsets, o[1][dy+1] row offsets, o[2][dz+1] plane offsets
    __device__ __forceinline__ long long at(int dx, int dy, int dz) const { return o[0][dx + 1] + o[1][dy + 1] + o[2][dz + 1]; }
};
__device__ __forceinline__ Nbr neighbours(long long n, int nx, int ny, int nz) {
    const int x = int(n % nx), y = int((n / nx) % ny), z = int(n / ((long long)nx * ny));
    Nbr b;
    b.o[0][0] = x == 0 ? nx - 1 : x - 1; b.o[0][1] = x; b.o[0][2] = x == nx - 1 ? 0 : x + 1;
    b.o[1][0] = (long long)nx * (y == 0 ? ny - 1 : y - 1); b.o[1][1] = (long long)nx * y; b.o[1][2] = (long long)nx * (y == ny - 1 ? 0 : y + 1);
    const long long pl = (long long)nx * ny;
    b.o[2][0] = pl * (z == 0 ? nz - 1 : z - 1); b.o[2][1] = pl * z; b.o[2][2] = pl * (z == nz - 1 ? 0 : z + 1);
    return b;
}

// The step-path kernels of the two-pass formulation run one thread block per ROW_BX consecutive x of one (y, z) row: no integer
// division, the y / z wrap is block-uniform, and consecutive blocks sweep memory in order (a linear sweep moves 6.7-6.9 TB/s on
// B200 where a march of tile columns moves 6.3: profiles/r2_probes.md).  grid = row_grid(): ny, nz <= 65535 (checked in lb_create).
constexpr int ROW_BX = 128;
__device__ __forceinline__ bool row_node(long long& n, Nbr& b, int& x, int& y, int& z, int nx, int ny, int nz) {
    x = blockIdx.x * ROW_BX + threadIdx.x; y = blockIdx.y; z = blockIdx.z;
    if (x >= nx) return false;
    b.o[0][0] = x == 0 ? nx - 1 : x - 1; b.o[0][1] = x; b.o[0][2] = x == nx - 1 ? 0 : x + 1;
    b.o[1][0] = (long long)nx * (y == 0 ? ny - 1 : y - 1); b.o[1][1] = (long long)nx * y; b.o[1][2] = (long long)nx * (y == ny - 1 ? 0 : y + 1);
    const long long pl = (long long)nx * ny;
    b.o[2][0] = pl * (z == 0 ? nz - 1 : z - 1); b.o[2][1] = pl * z; b.o[2][2] = pl * (z == nz - 1 ? 0 : z + 1);
    n = b.o[2][1] + b.o[1][1] + x;
    return true;
}

// the 19 populations of component k arriving at fluid node n: f_i(x) = h_i(x - c_i) (Eq. 5), or
// h_opp(i)(x) when x - c_i is solid (halfway bounce-back, Eq. 23-24 with u_b = 0).  lk = links[n].
template <typename T>
__device__ __forceinline__ void pull19(const T* __restrict__ h, long long NP, int k, long long n, const Nbr& b, unsigned lk, T (&fk)[Q]) {
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        const bool bounce = i > 0 && (lk >> dir_opp(i) & 1u);
        fk[i] = bounce ? plane(h, NP, k, dir_opp(i))[n] : plane(h, NP, k, i)[b.at(-dir_cx(i), -dir_cy(i), -dir_cz(i))];
    }
}

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

// f (streamed populations at their nodes) -> h-state: h_j(y) = f_j(y + c_j), or f_opp(j)(y) when
// y + c_j is solid (so that pulling h gives back exactly f).  Solid nodes hold 0.  links may be NULL.
template <typename T>
__global__ void __launch_bounds__(256) k_unstream(const T* __restrict__ f, T* __restrict__ h, const unsigned* __restrict__ links,
                                                  long long NP, int nx, int ny, int nz) {
    const long long N = (long long)nx * ny * nz;
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= N) return;
    const unsigned lk = links ? links[n] : 0u;
    const Nbr b = neighbours(n, nx, ny, nz);
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
        for (int j = 0; j < Q; ++j) {
            T v;
            if (lk & SOLID_BIT) v = T(0);
            else if (j > 0 && (lk >> j & 1u)) v = plane(f, NP, k, dir_opp(j))[n];
            else v = plane(f, NP, k, j)[b.at(dir_cx(j), dir_cy(j), dir_cz(j))];
            plane(h, NP, k, j)[n] = v;
        }
}

// h-state -> f: the streaming step itself (Eq. 5 / Eq. 23-24), written out for the getters.
template <typename T>
__global__ void __launch_bounds__(256) k_stream(const T* __restrict__ h, T* __restrict__ f, const unsigned* __restrict__ links,
                                                long long NP, int nx, int ny, int nz) {
    const long long N = (long long)nx * ny * nz;
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= N) return;
    const unsigned lk = links ? links[n] : 0u;
    const Nbr b = neighbours(n, nx, ny, nz);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        T fk[Q];
        if (lk & SOLID_BIT) {
#pragma unroll
            for (int i = 0; i < Q; ++i) fk[i] = T(0);
        } else {
            pull19<T>(h, NP, k, n, b, lk, fk);
        }
#pragma unroll
        for (int i = 0; i < Q; ++i) plane(f, NP, k, i)[n] = fk[i];
    }
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
__global__ void k_moments_out(const T* __restrict__ h, const unsigned* __restrict__ links, long long NP,
                              int nx, int ny, int nz, long long n0, long long cnt,
                              double* __restrict__ o_rr, double* __restrict__ o_rb, double* __restrict__ o_ux,
                              double* __restrict__ o_uy, double* __restrict__ o_uz) {
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= cnt) return;
    const long long n = n0 + t;
    const unsigned lk = links ? links[n] : 0u;
    T r[2] = {T(0), T(0)}, jx = T(0), jy = T(0), jz = T(0);
    if (!(lk & SOLID_BIT)) {
        const Nbr b = neighbours(n, nx, ny, nz);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            T fk[Q];
            pull19<T>(h, NP, k, n, b, lk, fk);
            T ax, ay, az;
            moments19<T>(fk, r[k], ax, ay, az);
            jx += ax; jy += ay; jz += az;
        }
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
__global__ void __launch_bounds__(256) k_diag_partial(const T* __restrict__ h, const unsigned* __restrict__ links, long long NP,
                                                      int nx, int ny, int nz, double* __restrict__ part) {
    const long long N = (long long)nx * ny * nz;
    double acc[5] = {0, 0, 0, 0, 0};
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < N; n += (long long)gridDim.x * blockDim.x) {
        const unsigned lk = links ? links[n] : 0u;
        if (lk & SOLID_BIT) continue;
        const Nbr b = neighbours(n, nx, ny, nz);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            T fk[Q];
            pull19<T>(h, NP, k, n, b, lk, fk);
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
// pass 1: rho^k(x,t) = sum_i f_i^k(x,t) (Eq. 6) with f pulled from the h-state.  Solid nodes report 0.
// Also the initialiser of the one-pass kernel's density arrays (rho_in = the whole sum, edge arrays 0).
template <typename T>
__global__ void __launch_bounds__(ROW_BX) k_density(const T* __restrict__ h, const unsigned* __restrict__ links, long long NP,
                                                    int nx, int ny, int nz, T* __restrict__ rho) {
    long long n; Nbr b; int x, y, z;
    if (!row_node(n, b, x, y, z, nx, ny, nz)) return;
    const unsigned lk = links ? links[n] : 0u;
    T r[2] = {T(0), T(0)};
    if (!(lk & SOLID_BIT)) {
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            T fk[Q];
            pull19<T>(h, NP, k, n, b, lk, fk);
            T ax, ay, az;
            moments19<T>(fk, r[k], ax, ay, az);
        }
    }
    rho[n] = r[0];
    rho[NP + n] = r[1];
}

// pass 2: pull (streaming + bounce-back of the previous step), Shan-Chen force, BGK collision with
// forcing; the post-collision values are written aligned, to be pulled by the next step.
template <typename T, bool HAS_SOLID>
__global__ void __launch_bounds__(ROW_BX) k_collide_pull(const T* __restrict__ h, T* __restrict__ g,
                                                         const T* __restrict__ rho, const unsigned* __restrict__ links,
                                                         long long NP, int nx, int ny, int nz,
                                                         T om_r, T om_b, T G) {
    long long n; Nbr b; int x, y, z;
    if (!row_node(n, b, x, y, z, nx, ny, nz)) return;
    unsigned lk = 0;
    if (HAS_SOLID) {
        lk = links[n];
        if (lk & SOLID_BIT) return;              // no computation inside a particle
    }
    T fr[Q], fb[Q];
    pull19<T>(h, NP, 0, n, b, lk, fr);
    pull19<T>(h, NP, 1, n, b, lk, fb);
    T rr, rb, jrx, jry, jrz, jbx, jby, jbz;
    moments19<T>(fr, rr, jrx, jry, jrz);
    moments19<T>(fb, rb, jbx, jby, jbz);
    const T den = om_r * rr + om_b * rb;                            // S4
    const T inv = den != T(0) ? T(1) / den : T(0);
    const T ux = (om_r * jrx + om_b * jbx) * inv, uy = (om_r * jry + om_b * jby) * inv, uz = (om_r * jrz + om_b * jbz) * inv;
    // du^k = -G sum_i w_i rho^kbar(x+c_i) c_i  (S2, S3, S6); solids report rho = 0 (S7)
    T gr[3] = {T(0), T(0), T(0)}, gb[3] = {T(0), T(0), T(0)};      // gradients of rho_b (acts on red) and rho_r (on blue)
#pragma unroll
    for (int p = 0; p < 9; ++p) {
        const long long np = b.at(pair_cx(p), pair_cy(p), pair_cz(p)), nm = b.at(-pair_cx(p), -pair_cy(p), -pair_cz(p));
        const T db = w_pair<T>(p) * (rho[NP + np] - rho[NP + nm]);
        const T dr = w_pair<T>(p) * (rho[np] - rho[nm]);
        if (pair_cx(p)) { gr[0] += T(pair_cx(p)) * db; gb[0] += T(pair_cx(p)) * dr; }
        if (pair_cy(p)) { gr[1] += T(pair_cy(p)) * db; gb[1] += T(pair_cy(p)) * dr; }
        if (pair_cz(p)) { gr[2] += T(pair_cz(p)) * db; gb[2] += T(pair_cz(p)) * dr; }
    }
    collide19<T>(fr, rr, T(1) - om_r, ux, uy, uz, ux - G * gr[0], uy - G * gr[1], uz - G * gr[2]);
    collide19<T>(fb, rb, T(1) - om_b, ux, uy, uz, ux - G * gb[0], uy - G * gb[1], uz - G * gb[2]);
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        plane(g, NP, 0, i)[n] = fr[i];
        plane(g, NP, 1, i)[n] = fb[i];
    }
}

// ----------------------------------------------------------------------------------------
// later operators on the two-pass path: colour-gradient collision and moving walls
// ----------------------------------------------------------------------------------------
// pass 1 of the colour-gradient step: Theta = (rho^1 - rho^2) / (rho^1 + rho^2); 0 on solid and empty nodes (reading C1)
template <typename T>
__global__ void __launch_bounds__(ROW_BX) k_phase_field(const T* __restrict__ h, const unsigned* __restrict__ links, long long NP,
                                                        int nx, int ny, int nz, T* __restrict__ theta) {
    long long n; Nbr b; int x, y, z;
    if (!row_node(n, b, x, y, z, nx, ny, nz)) return;
    const unsigned lk = links ? links[n] : 0u;
    T th = T(0);
    if (!(lk & SOLID_BIT)) {
        T r[2];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            T fk[Q], ax, ay, az;
            pull19<T>(h, NP, k, n, b, lk, fk);
            moments19<T>(fk, r[k], ax, ay, az);
        }
        const T rt = r[0] + r[1];
        if (rt != T(0)) th = (r[0] - r[1]) / rt;
    }
    theta[n] = th;
}

struct SphereView {
    const double* c; const double* v; const double* w;     // [p][3] centres, velocities, angular velocities
    double* F; double* T;                                  // [p][3] accumulators of this step (fp64 for both dtypes)
    const int* pid;                                        // sphere of every solid node, -1 = a solid at rest that is no sphere
};

// B_i of PAPER.md:393-398
template <typename T> __host__ __device__ constexpr T b_rest() { return T(-2.0 / 9.0); }
template <typename T> __host__ __device__ constexpr T b_pair(int p) { return p < 3 ? T(1.0 / 54.0) : T(1.0 / 27.0); }

// pass 2 for both collision operators, with optional moving walls.
//   MODEL 0: Shan-Chen as k_collide_pull (aux = rho[2][NP]).
//   MODEL 1: colour gradient (readings C1-C6 of DESIGN.md section 3), aux = Theta[NP]:
//            u by Eq. 7, omega from the mean viscosity, BGK (Eq. 9-10), perturbation (Eq. 17, A by Eq. 19),
//            recolouring (Eq. 20-21).
//   MOVING:  a link i into a sphere with velocity u_b = v_p + r_b x omega_p (Eq. 22) returns f*_i - 2 rho^k w_i u_b.c_i / c_s^2
//            (Eq. 24) and hands c_i (f*_i + that) to the sphere (Eq. 25-27; readings M1-M4).  The value is stored where the
//            plain bounce-back finds it: in the node's own slot i of the post-collision state.
template <typename T, int MODEL, bool MOVING>
__global__ void __launch_bounds__(ROW_BX) k_collide_next(const T* __restrict__ h, T* __restrict__ g, const T* __restrict__ aux,
                                                      const unsigned* __restrict__ links, long long NP, int nx, int ny, int nz,
                                                      T om_r, T om_b, T G, T sigma, T beta, T nu_r, T nu_b, SphereView sp) {
    long long n; Nbr b; int x, y, z;
    if (!row_node(n, b, x, y, z, nx, ny, nz)) return;
    const unsigned lk = links ? links[n] : 0u;
    if (lk & SOLID_BIT) return;
    T fr[Q], fb[Q];
    pull19<T>(h, NP, 0, n, b, lk, fr);
    pull19<T>(h, NP, 1, n, b, lk, fb);
    T rr, rb, jrx, jry, jrz, jbx, jby, jbz;
    moments19<T>(fr, rr, jrx, jry, jrz);
    moments19<T>(fb, rb, jbx, jby, jbz);
    if (MODEL == 0) {
        const T den = om_r * rr + om_b * rb;
        const T inv = den != T(0) ? T(1) / den : T(0);
        const T ux = (om_r * jrx + om_b * jbx) * inv, uy = (om_r * jry + om_b * jby) * inv, uz = (om_r * jrz + om_b * jbz) * inv;
        T gr[3] = {T(0), T(0), T(0)}, gb[3] = {T(0), T(0), T(0)};
#pragma unroll
        for (int p = 0; p < 9; ++p) {
            const long long np = b.at(pair_cx(p), pair_cy(p), pair_cz(p)), nm = b.at(-pair_cx(p), -pair_cy(p), -pair_cz(p));
            const T db = w_pair<T>(p) * (aux[NP + np] - aux[NP + nm]);
            const T dr = w_pair<T>(p) * (aux[np] - aux[nm]);
            if (pair_cx(p)) { gr[0] += T(pair_cx(p)) * db; gb[0] += T(pair_cx(p)) * dr; }
            if (pair_cy(p)) { gr[1] += T(pair_cy(p)) * db; gb[1] += T(pair_cy(p)) * dr; }
            if (pair_cz(p)) { gr[2] += T(pair_cz(p)) * db; gb[2] += T(pair_cz(p)) * dr; }
        }
        collide19<T>(fr, rr, T(1) - om_r, ux, uy, uz, ux - G * gr[0], uy - G * gr[1], uz - G * gr[2]);
        collide19<T>(fb, rb, T(1) - om_b, ux, uy, uz, ux - G * gb[0], uy - G * gb[1], uz - G * gb[2]);
    } else {
        const T rt = rr + rb;
        if (rt == T(0)) {                                                   // reading C6
#pragma unroll
            for (int i = 0; i < Q; ++i) { fr[i] = T(0); fb[i] = T(0); }
        } else {
            const T irt = T(1) / rt;
            const T ux = (jrx + jbx) * irt, uy = (jry + jby) * irt, uz = (jrz + jbz) * irt;      // Eq. 7
            const T xr = rr * irt, xb = rb * irt;
            const T om = T(2) / (T(6) / (xr / nu_r + xb / nu_b) + T(1));                       // PAPER.md:336, reading C2
            const T A = T(2.25) * sigma * om;                                                  // Eq. 19
            T gx = T(0), gy = T(0), gz = T(0);                                                 // grad Theta, reading C1
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const T d = w_pair<T>(p) * (aux[b.at(pair_cx(p), pair_cy(p), pair_cz(p))] - aux[b.at(-pair_cx(p), -pair_cy(p), -pair_cz(p))]);
                if (pair_cx(p)) gx += T(pair_cx(p)) * d;
                if (pair_cy(p)) gy += T(pair_cy(p)) * d;
                if (pair_cz(p)) gz += T(pair_cz(p)) * d;
            }
            gx *= T(3); gy *= T(3); gz *= T(3);
            const T g2 = gx * gx + gy * gy + gz * gz;
            const T gn = sqrt(g2);
            const T ig2 = g2 != T(0) ? T(1) / g2 : T(0), ign = g2 != T(0) ? T(1) / gn : T(0);
            const T amp = T(0.5) * A * gn;                                                     // (A / 2) |grad|, 0 without a gradient
            const T rc = beta * xr * xb * rt;                                                  // beta rho^1 rho^2 / rho^2 times rho of f^{eq,0}
            const T a0 = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
            {   // rest direction: cos(phi) = 0
                const T fstar = (T(1) - om) * (fr[0] + fb[0]) + om * w_rest<T>() * rt * a0 + T(2) * amp * (-b_rest<T>());
                fr[0] = xr * fstar; fb[0] = xb * fstar;
            }
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const T cu = cdot<T>(p, ux, uy, uz), cg = cdot<T>(p, gx, gy, gz);
                const T wr = w_pair<T>(p) * rt;
                const T s0 = a0 + T(4.5) * cu * cu;
                const T pert = T(2) * amp * (w_pair<T>(p) * cg * cg * ig2 - b_pair<T>(p));      // both components' Eq. 17, same for i and opp(i)
                const T recol = rc * w_pair<T>(p) * cg * ign * (p < 3 ? T(1) : T(0.70710678118654752440));   // cos(phi_i) = c_i.grad / (|c_i| |grad|)
                const T f1 = (T(1) - om) * (fr[2 * p + 1] + fb[2 * p + 1]) + om * wr * (s0 + T(3) * cu) + pert;
                const T f2 = (T(1) - om) * (fr[2 * p + 2] + fb[2 * p + 2]) + om * wr * (s0 - T(3) * cu) + pert;
                fr[2 * p + 1] = xr * f1 + recol; fb[2 * p + 1] = xb * f1 - recol;               // Eq. 20-21
                fr[2 * p + 2] = xr * f2 - recol; fb[2 * p + 2] = xb * f2 + recol;
            }
        }
    }
    if (MOVING && (lk & 0x7FFFEu)) {
        // a loop over the links that exist (few nodes have any, and those few a handful): compact code instead of 18 unrolled copies.
        // The two values of a link are exchanged with the register arrays through a switch-free select chain on the direction.
        // Force and torque of this node's links are added up in registers and handed to the sphere's sums once per node (the links of a
        // node nearly always end in one sphere): 6 atomics per node instead of 6 per link.
        int pcur = -1;
        double Fa[3] = {0, 0, 0}, Ta[3] = {0, 0, 0};
        auto flush = [&]() {
            if (pcur < 0) return;
#pragma unroll
            for (int a_ = 0; a_ < 3; ++a_) {
                if (Fa[a_] != 0.0) atomicAdd(sp.F + 3 * pcur + a_, Fa[a_]);
                if (Ta[a_] != 0.0) atomicAdd(sp.T + 3 * pcur + a_, Ta[a_]);
                Fa[a_] = 0.0; Ta[a_] = 0.0;
            }
        };
        for (unsigned m = lk & 0x7FFFEu; m; m &= m - 1) {
            const int i = __ffs(int(m)) - 1;
            const int cx = dir_cx(i), cy = dir_cy(i), cz = dir_cz(i);
            const int p = sp.pid[b.at(cx, cy, cz)];
            if (p < 0) continue;
            if (p != pcur) { flush(); pcur = p; }
            double rbv[3] = {x + 0.5 * cx - sp.c[3 * p], y + 0.5 * cy - sp.c[3 * p + 1], z + 0.5 * cz - sp.c[3 * p + 2]};
            // minimum image: r - n floor(r / n + 1/2) for |r| < n, without the divisions (this loop runs in most warps: nearly every
            // 128-node row passes a sphere, and the warp waits for the lane with the most links)
            const double hx_ = 0.5 * nx, hy_ = 0.5 * ny, hz_ = 0.5 * nz;
            rbv[0] -= rbv[0] >= hx_ ? double(nx) : (rbv[0] < -hx_ ? -double(nx) : 0.0);
            rbv[1] -= rbv[1] >= hy_ ? double(ny) : (rbv[1] < -hy_ ? -double(ny) : 0.0);
            rbv[2] -= rbv[2] >= hz_ ? double(nz) : (rbv[2] < -hz_ ? -double(nz) : 0.0);
            const double ub[3] = {sp.v[3 * p] + (rbv[1] * sp.w[3 * p + 2] - rbv[2] * sp.w[3 * p + 1]),      // Eq. 22 as printed
                                  sp.v[3 * p + 1] + (rbv[2] * sp.w[3 * p] - rbv[0] * sp.w[3 * p + 2]),
                                  sp.v[3 * p + 2] + (rbv[0] * sp.w[3 * p + 1] - rbv[1] * sp.w[3 * p])};
            const T wi = i < 7 ? T(1.0 / 18.0) : T(1.0 / 36.0);
            const T ubi = T(3) * T(ub[0] * cx + ub[1] * cy + ub[2] * cz);
            T fri = T(0), fbi = T(0);
#pragma unroll
            for (int q = 1; q < Q; ++q) if (q == i) { fri = fr[q]; fbi = fb[q]; }
            const T br = fri - T(2) * rr * wi * ubi, bb = fbi - T(2) * rb * wi * ubi;                  // Eq. 24
            const double mm = (double(fri) + double(br)) + (double(fbi) + double(bb));                 // momentum handed over along c_i
#pragma unroll
            for (int q = 1; q < Q; ++q) if (q == i) { fr[q] = br; fb[q] = bb; }
            const double Fv[3] = {mm * cx, mm * cy, mm * cz};
            Fa[0] += Fv[0]; Fa[1] += Fv[1]; Fa[2] += Fv[2];
            Ta[0] += Fv[1] * rbv[2] - Fv[2] * rbv[1];                                                 // Eq. 27 as printed: F x r_b
            Ta[1] += Fv[2] * rbv[0] - Fv[0] * rbv[2];
            Ta[2] += Fv[0] * rbv[1] - Fv[1] * rbv[0];
        }
        flush();
    }
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        plane(g, NP, 0, i)[n] = fr[i];
        plane(g, NP, 1, i)[n] = fb[i];
    }
}

inline unsigned blocks_for(long long cnt, int bs) { return unsigned((cnt + bs - 1) / bs); }
inline dim3 row_grid(const lb_ctx* c) { return dim3(unsigned((c->nx + ROW_BX - 1) / ROW_BX), unsigned(c->ny), unsigned(c->nz)); }

bool onepass_ok(const lb_ctx* c) { return c->nx % OP_TX == 0 && c->ny % OP_TY == 0; }

// rho_*[rcur] := density of the state in f[cur] (rho_in = the whole sum, the edge arrays zero)
template <typename T>
int ensure_rho(lb_ctx* c) {
    if (c->rho_valid && c->rho_fmt == RHO_FULL) return LB_OK;
    c->rho_fmt = RHO_FULL;
    const int r = c->rcur;
    if (c->rho_x[r]) {
        CU(cudaMemsetAsync(c->rho_x[r], 0, size_t(2) * c->s_x * sizeof(T), c->stream));
        CU(cudaMemsetAsync(c->rho_y[r], 0, size_t(2) * c->s_y * sizeof(T), c->stream));
        CU(cudaMemsetAsync(c->rho_xy[r], 0, size_t(2) * c->s_xy * sizeof(T), c->stream));
    }
    k_density<T><<<row_grid(c), ROW_BX, 0, c->stream>>>(static_cast<const T*>(c->f[c->cur]), c->has_solid ? c->links : nullptr,
                                                               c->NP, c->nx, c->ny, c->nz, static_cast<T*>(c->rho_in[r]));
    c->launches++;
    CU(cudaGetLastError());
    c->rho_valid = true;
    return LB_OK;
}

template <typename T>
int step_twopass(lb_ctx* c) {
    c->rho_valid = false;                                   // this path keeps no density across steps
    const int rc = ensure_rho<T>(c);
    if (rc != LB_OK) return rc;
    const T* h = static_cast<const T*>(c->f[c->cur]);
    T* g = static_cast<T*>(c->f[c->cur ^ 1]);
    const T* rho = static_cast<const T*>(c->rho_in[c->rcur]);
    const dim3 nb = row_grid(c);
    const T om_r = T(1.0 / c->tau[0]), om_b = T(1.0 / c->tau[1]), G = T(c->G);
    if (c->has_solid)
        k_collide_pull<T, true><<<nb, ROW_BX, 0, c->stream>>>(h, g, rho, c->links, c->NP, c->nx, c->ny, c->nz, om_r, om_b, G);
    else
        k_collide_pull<T, false><<<nb, ROW_BX, 0, c->stream>>>(h, g, rho, nullptr, c->NP, c->nx, c->ny, c->nz, om_r, om_b, G);
    c->launches += 1;
    CU(cudaGetLastError());
    c->cur ^= 1;
    c->rho_valid = false;
    c->hx_valid = false;
    c->diag_fresh = false;
    return LB_OK;
}

SphereView sphere_view(const lb_ctx* c) {
    SphereView v;
    v.c = c->sph; v.v = c->sph + 3 * c->nsph; v.w = c->sph + 6 * c->nsph; v.F = c->sph + 9 * c->nsph; v.T = c->sph + 12 * c->nsph;
    v.pid = c->pid;
    return v;
}

// one step of the later operators: colour gradient and / or moving walls, any box shape
template <typename T>
int step_next(lb_ctx* c) {
    const T* h = static_cast<const T*>(c->f[c->cur]);
    T* g = static_cast<T*>(c->f[c->cur ^ 1]);
    T* aux = static_cast<T*>(c->rho_in[c->rcur]);
    const unsigned* lk = c->has_solid ? c->links : nullptr;
    const dim3 nb = row_grid(c);
    if (c->model == LB_MODEL_COLOUR_GRADIENT) k_phase_field<T><<<nb, ROW_BX, 0, c->stream>>>(h, lk, c->NP, c->nx, c->ny, c->nz, aux);
    else k_density<T><<<nb, ROW_BX, 0, c->stream>>>(h, lk, c->NP, c->nx, c->ny, c->nz, aux);
    const bool moving = c->nsph > 0;
    SphereView sp = {};
    if (moving) {
        sp = sphere_view(c);
        CU(cudaMemsetAsync(sp.F, 0, size_t(6) * c->nsph * sizeof(double), c->stream));
    }
    const T om_r = T(1.0 / c->tau[0]), om_b = T(1.0 / c->tau[1]), G = T(c->G), sg = T(c->sigma), be = T(c->beta);
    const T nu_r = T((c->tau[0] - 0.5) / 3.0), nu_b = T((c->tau[1] - 0.5) / 3.0);
#define LB_NEXT(MODEL, MOVING) k_collide_next<T, MODEL, MOVING><<<nb, ROW_BX, 0, c->stream>>>(h, g, aux, lk, c->NP, c->nx, c->ny, c->nz, om_r, om_b, G, sg, be, nu_r, nu_b, sp)
    if (c->model == LB_MODEL_COLOUR_GRADIENT) { if (moving) LB_NEXT(1, true); else LB_NEXT(1, false); }
    else { if (moving) LB_NEXT(0, true); else LB_NEXT(0, false); }
#undef LB_NEXT
    c->launches += 2;
    CU(cudaGetLastError());
    c->cur ^= 1;
    c->rho_valid = false;
    c->hx_valid = false;
    c->diag_fresh = false;
    return LB_OK;
}

template <typename T>
int zero_solids(lb_ctx* c, int buf) {
    k_zero_solids<T><<<blocks_for(c->N, 256), 256, 0, c->stream>>>(static_cast<T*>(c->f[buf]), c->NP, c->N, c->links);
    c->launches++;
    CU(cudaGetLastError());
    return LB_OK;
}

// f in the scratch buffer -> h-state in f[cur]; the scratch keeps zeros on solid nodes
template <typename T>
int unstream_scratch(lb_ctx* c) {
    k_unstream<T><<<blocks_for(c->N, 256), 256, 0, c->stream>>>(static_cast<const T*>(c->f[c->cur ^ 1]), static_cast<T*>(c->f[c->cur]),
                                                                c->has_solid ? c->links : nullptr, c->NP, c->nx, c->ny, c->nz);
    c->launches++;
    CU(cudaGetLastError());
    c->rho_valid = false;
    c->hx_valid = false;
    c->diag_fresh = false;
    return LB_OK;
}

// h-state -> f in the scratch buffer
template <typename T>
int stream_to_scratch(lb_ctx* c) {
    k_stream<T><<<blocks_for(c->N, 256), 256, 0, c->stream>>>(static_cast<const T*>(c->f[c->cur]), static_cast<T*>(c->f[c->cur ^ 1]),
                                                              c->has_solid ? c->links : nullptr, c->NP, c->nx, c->ny, c->nz);
    c->launches++;
    CU(cudaGetLastError());
    return LB_OK;
}

// ----------------------------------------------------------------------------------------
// one-pass time step (lb_onepass.cuh): boxes whose x, y sides are multiples of the 32 x 8 tile
// ----------------------------------------------------------------------------------------
constexpr int OP_RESIDENT_CTAS = 148 * 2;

// planes per CTA: every chunk re-collides 2 extra planes, so long chunks; but the grid should
// still be several waves of the resident CTAs.  lb_set_option(LB_OPT_ZC) overrides.
int onepass_zc(const lb_ctx* c) {
    if (c->zc_req >= 1) return c->zc_req < c->nz ? c->zc_req : c->nz;
    const long long tiles = (long long)(c->nx / OP_TX) * (c->ny / OP_TY);
    const long long chunks_wanted = (OP_RESIDENT_CTAS * 4 + tiles - 1) / (tiles > 0 ? tiles : 1);
    long long zc = c->nz / (chunks_wanted > 0 ? chunks_wanted : 1);
    if (zc > 128) zc = 128;
    if (zc < 16) zc = 16;
    if (zc > c->nz) zc = c->nz;
    for (long long d = zc; d >= (zc + 1) / 2; --d)
        if (c->nz % d == 0) return int(d);
    return int(zc);
}

template <typename T>
RhoView<T> rho_view(const lb_ctx* c, int r) {
    RhoView<T> v;
    v.in = static_cast<T*>(c->rho_in[r]); v.s_in = c->NP;
    v.x = static_cast<T*>(c->rho_x[r]); v.s_x = c->s_x;
    v.y = static_cast<T*>(c->rho_y[r]); v.s_y = c->s_y;
    v.xy = static_cast<T*>(c->rho_xy[r]); v.s_xy = c->s_xy;
    return v;
}

template <typename T, bool HAS_SOLID>
int launch_onepass(lb_ctx* c) {
    auto kern = k_step_pull<T, HAS_SOLID, OP_TX, OP_TY>;
    constexpr size_t smem = onepass_smem_bytes<T, OP_TX, OP_TY>();
    const dim3 grid(c->nx / OP_TX, c->ny / OP_TY, (c->nz + c->zc - 1) / c->zc);
    const T om_r = T(1.0 / c->tau[0]), om_b = T(1.0 / c->tau[1]), G = T(c->G);
    kern<<<grid, OP_TX * OP_TY, smem, c->stream>>>(static_cast<const T*>(c->f[c->cur]), static_cast<T*>(c->f[c->cur ^ 1]),
                                                   HAS_SOLID ? c->links : nullptr, rho_view<T>(c, c->rcur), rho_view<T>(c, c->rcur ^ 1),
                                                   c->NP, c->nx, c->ny, c->nz, c->zc, om_r, om_b, G);
    c->launches += 1;
    CU(cudaGetLastError());
    return LB_OK;
}

template <typename T>
int step_onepass(lb_ctx* c) {
    int rc = ensure_rho<T>(c);
    if (rc != LB_OK) return rc;
    rc = c->has_solid ? launch_onepass<T, true>(c) : launch_onepass<T, false>(c);
    if (rc != LB_OK) return rc;
    c->cur ^= 1;
    c->rcur ^= 1;                                           // the kernel wrote rho(t+1)
    c->hx_valid = false;
    c->diag_fresh = false;
    return LB_OK;
}

// ----------------------------------------------------------------------------------------
// TMA-staged one-pass time step (lb_tma.cuh): same boxes, same density arrays as the one-pass kernel
// ----------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// tensor maps over the population buffers: dims (x, y, z, plane), one box = one tile row block of one plane
bool make_tmaps(lb_ctx* c) {
    EncodeTiledFn enc = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", reinterpret_cast<void**>(&enc), cudaEnableDefault, &qr) != cudaSuccess || !enc) {
        cudaGetLastError();
        return false;
    }
    const cuuint64_t es = esize(c);
    const cuuint64_t gdim[4] = {cuuint64_t(c->nx), cuuint64_t(c->ny), cuuint64_t(c->nz), cuuint64_t(NPOP)};
    const cuuint64_t gstr[3] = {cuuint64_t(c->nx) * es, cuuint64_t(c->nx) * c->ny * es, cuuint64_t(c->NP) * es};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUtensorMapDataType dt = c->dtype == LB_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    for (int b = 0; b < 2; ++b)
        for (int w = 0; w < 3; ++w) {
            const cuuint32_t pad = cuuint32_t(16 / int(es));
            const cuuint32_t box[4] = {w == 0 ? cuuint32_t(OP_TX) : (w == 1 ? OP_TX + pad : pad), cuuint32_t(OP_TY), 1, 2};   // both components (pop_plane)
            if (enc(&c->tmap[b][w], dt, 4, c->f[b], gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                    CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
                return false;
        }
    // x-halo arrays: dims (y', tile_x, z, plane 2 j + k), one box = the TY rows of one tile, both components
    const cuuint64_t ntx = cuuint64_t(c->nx / OP_TX);
    const cuuint64_t hdim[4] = {cuuint64_t(c->ny), ntx, cuuint64_t(c->nz), cuuint64_t(2 * NHALO)};
    const cuuint64_t hstr[3] = {cuuint64_t(c->ny) * es, cuuint64_t(c->ny) * ntx * es, cuuint64_t(c->ny) * ntx * c->nz * es};
    const cuuint32_t hbox[4] = {cuuint32_t(OP_TY), 1, 1, 2};
    for (int b = 0; b < 2; ++b)
        if (enc(&c->tmap_hx[b], dt, 4, c->hx[b], hdim, hstr, hbox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    return true;
}

// Grid of k_step_tma / k_step_node (chunk_range in lb_tma.cuh): nz / zc_tma chunks per tile column; when the planes per CTA were
// left to the library (and the kernel keeps no per-CTA sums), the last tile columns, from col_split on, are cut into one chunk
// more so that the number of working CTAs is a multiple of the SM count.
dim3 tma_grid(const lb_ctx* c, bool allow_balance, int& col_split) {
    const int ntx = c->nx / OP_TX, nty = c->ny / OP_TY, nchunk = c->nz / c->zc_tma;
    col_split = ntx * nty;
    if (allow_balance && c->zc_req == 0 && c->balance) {
        int sms = 148;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
        const long long total = (long long)ntx * nty * nchunk;
        const int more = int((sms - total % sms) % sms);               // CTAs missing to the next multiple: one more per tile column
        if (total > sms && more >= 1 && more < ntx * nty && c->nz / (nchunk + 1) >= 8) col_split = ntx * nty - more;
    }
    return dim3(ntx, nty, col_split < ntx * nty ? nchunk + 1 : nchunk);
}

int ensure_diag_buf(lb_ctx* c, long long ncta) {
    if (c->diag_cta && c->diag_cta_cap >= ncta) return LB_OK;
    CU(cudaStreamSynchronize(c->stream));
    cudaFree(c->diag_cta);
    c->diag_cta = nullptr;
    CU(cudaMalloc(&c->diag_cta, size_t(ncta) * 5 * sizeof(double)));
    c->diag_cta_cap = ncta;
    return LB_OK;
}

template <typename T, bool HAS_SOLID, bool DIAG, int MODEL = 0>
int launch_tma(lb_ctx* c) {
    auto kern = k_step_tma<T, HAS_SOLID, OP_TY, DIAG, MODEL>;
    constexpr size_t smem = TmaLayout<T, OP_TY>::BYTES;
    int col_split;
    const dim3 grid(tma_grid(c, !DIAG, col_split));
    const T om_r = T(1.0 / c->tau[0]), om_b = T(1.0 / c->tau[1]), G = T(MODEL == 1 ? c->sigma : c->G);
    if (DIAG) {
        const long long ncta = (long long)grid.x * grid.y * grid.z;
        const int rc = ensure_diag_buf(c, ncta);
        if (rc != LB_OK) return rc;
        c->diag_ncta = ncta;
    }
    kern<<<grid, 2 * OP_TX * OP_TY + 128, smem, c->stream>>>(c->tmap[c->cur][0], c->tmap[c->cur][1], c->tmap[c->cur][2], static_cast<const T*>(c->f[c->cur]),
                                                           static_cast<T*>(c->f[c->cur ^ 1]), HAS_SOLID ? c->links : nullptr,
                                                           rho_view<T>(c, c->rcur), rho_view<T>(c, c->rcur ^ 1), c->NP, c->nx, c->ny, c->nz,
                                                           c->zc_tma, om_r, om_b, G, c->diag_cta, T(c->beta), col_split);
    c->launches += 1;
    CU(cudaGetLastError());
    return LB_OK;
}

template <typename T>
int step_tma(lb_ctx* c) {
    int rc = ensure_rho<T>(c);
    if (rc != LB_OK) return rc;
    const bool cg = c->model == LB_MODEL_COLOUR_GRADIENT;   // (effective_kernel sends colour gradient with solids down the two-pass path)
    const bool diag = c->diag_mode && !c->has_solid && !cg; // with bounce-back the walls take momentum: the separate pass does it
    rc = cg ? launch_tma<T, false, false, 1>(c)
            : (c->has_solid ? launch_tma<T, true, false>(c) : (diag ? launch_tma<T, false, true>(c) : launch_tma<T, false, false>(c)));
    if (rc != LB_OK) return rc;
    c->cur ^= 1;
    c->rcur ^= 1;                                           // the kernel wrote rho(t+1)
    c->hx_valid = false;
    c->diag_fresh = diag;
    return LB_OK;
}

// ----------------------------------------------------------------------------------------
// one thread per node (lb_node.cuh): same state and arrays as the TMA kernel, boxes without solid nodes
// ----------------------------------------------------------------------------------------
template <typename T>
int step_node(lb_ctx* c) {
    int rc = ensure_rho<T>(c);
    if (rc != LB_OK) return rc;
    const bool cg = c->model == LB_MODEL_COLOUR_GRADIENT;
    const bool diag = c->diag_mode && !cg;
    auto kern = cg ? k_step_node<T, OP_TY, 1, false> : (diag ? k_step_node<T, OP_TY, 0, true> : k_step_node<T, OP_TY, 0, false>);
    constexpr size_t smem = TmaLayout<T, OP_TY>::BYTES;
    int col_split;
    const dim3 grid(tma_grid(c, !diag, col_split));
    if (diag) {
        const long long ncta = (long long)grid.x * grid.y * grid.z;
        rc = ensure_diag_buf(c, ncta);
        if (rc != LB_OK) return rc;
        c->diag_ncta = ncta;
    }
    kern<<<grid, OP_TX * OP_TY + 128, smem, c->stream>>>(c->tmap[c->cur][0], c->tmap[c->cur][1], c->tmap[c->cur][2], static_cast<const T*>(c->f[c->cur]),
                                                       static_cast<T*>(c->f[c->cur ^ 1]), rho_view<T>(c, c->rcur), rho_view<T>(c, c->rcur ^ 1),
                                                       c->NP, c->nx, c->ny, c->nz, c->zc_tma, T(1.0 / c->tau[0]), T(1.0 / c->tau[1]), T(cg ? c->sigma : c->G), col_split, T(c->beta), c->diag_cta);
    c->launches += 1;
    CU(cudaGetLastError());
    c->cur ^= 1;
    c->rcur ^= 1;
    c->hx_valid = false;
    c->diag_fresh = diag;
    return LB_OK;
}

// ----------------------------------------------------------------------------------------
// halo kernel (lb_halo.cuh): boxes without solid nodes
// ----------------------------------------------------------------------------------------
template <typename T>
EdgeView<T> edge_view(const lb_ctx* c, int r) {
    EdgeView<T> v;
    v.er = static_cast<T*>(c->rho_er[r]); v.ec = static_cast<T*>(c->rho_ec[r]);
    v.x = static_cast<T*>(c->rho_x[r]); v.s_x = c->s_x;
    v.y = static_cast<T*>(c->rho_y[r]); v.s_y = c->s_y;
    v.xy = static_cast<T*>(c->rho_xy[r]); v.s_xy = c->s_xy;
    return v;
}

// the frame-density arrays [rcur] and the x-halo copies hx[cur] of the state in f[cur]
template <typename T>
int ensure_halo_state(lb_ctx* c) {
    if (!(c->rho_valid && c->rho_fmt == RHO_EDGE)) {
        const int r = c->rcur;
        CU(cudaMemsetAsync(c->rho_x[r], 0, size_t(2) * c->s_x * sizeof(T), c->stream));
        CU(cudaMemsetAsync(c->rho_y[r], 0, size_t(2) * c->s_y * sizeof(T), c->stream));
        CU(cudaMemsetAsync(c->rho_xy[r], 0, size_t(2) * c->s_xy * sizeof(T), c->stream));
        k_density<T><<<row_grid(c), ROW_BX, 0, c->stream>>>(static_cast<const T*>(c->f[c->cur]), nullptr, c->NP, c->nx, c->ny, c->nz,
                                                                   static_cast<T*>(c->rho_in[r]));
        k_edges_from_rho<T><<<blocks_for(c->N, 256), 256, 0, c->stream>>>(static_cast<const T*>(c->rho_in[r]), c->NP, edge_view<T>(c, r),
                                                                          c->nx, c->ny, c->nz, OP_TY);
        c->launches += 2;
        CU(cudaGetLastError());
        c->rho_valid = true;
        c->rho_fmt = RHO_EDGE;
    }
    if (!c->hx_valid) {
        k_fill_xhalo<T><<<blocks_for(c->hx_elems, 256), 256, 0, c->stream>>>(static_cast<const T*>(c->f[c->cur]), static_cast<T*>(c->hx[c->cur]),
                                                                             c->NP, c->nx, c->ny, c->nz);
        c->launches++;
        CU(cudaGetLastError());
        c->hx_valid = true;
    }
    return LB_OK;
}


template <typename T, bool DIAG>
int launch_halo(lb_ctx* c) {
    auto kern = k_step_halo<T, DIAG, OP_TY>;
    constexpr size_t smem = HaloLayout<T, OP_TY>::template bytes<DIAG>();
    const dim3 grid(c->nx / OP_TX, c->ny / OP_TY, c->nz / c->zc_tma);
    const T om_r = T(1.0 / c->tau[0]), om_b = T(1.0 / c->tau[1]), G = T(c->G);
    if (DIAG) {
        const long long ncta = (long long)grid.x * grid.y * grid.z;
        const int rc = ensure_diag_buf(c, ncta);
        if (rc != LB_OK) return rc;
        c->diag_ncta = ncta;
    }
    kern<<<grid, 2 * OP_TX * OP_TY + 128, smem, c->stream>>>(c->tmap[c->cur][0], c->tmap_hx[c->cur], static_cast<const T*>(c->f[c->cur]),
                                                           static_cast<T*>(c->f[c->cur ^ 1]), static_cast<T*>(c->hx[c->cur ^ 1]),
                                                           edge_view<T>(c, c->rcur), edge_view<T>(c, c->rcur ^ 1), c->diag_cta,
                                                           c->NP, c->nx, c->ny, c->nz, c->zc_tma, om_r, om_b, G);
    c->launches += 1;
    CU(cudaGetLastError());
    return LB_OK;
}

template <typename T>
int step_halo(lb_ctx* c) {
    int rc = ensure_halo_state<T>(c);
    if (rc != LB_OK) return rc;
    rc = c->diag_mode ? launch_halo<T, true>(c) : launch_halo<T, false>(c);
    if (rc != LB_OK) return rc;
    c->cur ^= 1;
    c->rcur ^= 1;                                           // the kernel wrote the frame densities of t+1 ...
    c->diag_fresh = c->diag_mode != 0;                      // ... the x-halo copies of the new populations, and (DIAG) their sums
    return LB_OK;
}

// The one-pass kernels use more dynamic shared memory than the default limit: opt in once per context (the attribute is
// per device and per function; setting it again is harmless).
template <typename T>
int configure_onepass_kernels() {
    CU(cudaFuncSetAttribute(k_step_pull<T, false, OP_TX, OP_TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(onepass_smem_bytes<T, OP_TX, OP_TY>())));
    CU(cudaFuncSetAttribute(k_step_pull<T, true, OP_TX, OP_TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(onepass_smem_bytes<T, OP_TX, OP_TY>())));
    CU(cudaFuncSetAttribute(k_step_tma<T, false, OP_TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(TmaLayout<T, OP_TY>::BYTES)));
    CU(cudaFuncSetAttribute(k_step_tma<T, true, OP_TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(TmaLayout<T, OP_TY>::BYTES)));
    CU(cudaFuncSetAttribute(k_step_tma<T, false, OP_TY, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(TmaLayout<T, OP_TY>::BYTES)));
    CU(cudaFuncSetAttribute(k_step_tma<T, false, OP_TY, false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(TmaLayout<T, OP_TY>::BYTES)));
    CU(cudaFuncSetAttribute(k_step_node<T, OP_TY, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(TmaLayout<T, OP_TY>::BYTES)));
    CU(cudaFuncSetAttribute(k_step_node<T, OP_TY, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(TmaLayout<T, OP_TY>::BYTES)));
    CU(cudaFuncSetAttribute(k_step_node<T, OP_TY, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(TmaLayout<T, OP_TY>::BYTES)));
    CU(cudaFuncSetAttribute(k_step_halo<T, false, OP_TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(HaloLayout<T, OP_TY>::template bytes<false>())));
    CU(cudaFuncSetAttribute(k_step_halo<T, true, OP_TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(HaloLayout<T, OP_TY>::template bytes<true>())));
    return LB_OK;
}

// planes per CTA of the TMA kernels: every chunk re-collides 2 extra planes and fills its pipeline (short chunks cost), and the last
// CTAs of a launch leave SMs idle for about half a CTA's run time (long chunks cost).  time(zc) ~ (zc + 4) * (max(1, waves) + 0.5),
// waves = CTAs / SMs: reproduces the measured order at 256^3 (zc 64: 1.99 ms, 32: 2.04, 128: 2.06), 512^3 (128: 16.08 ms, 64: 16.16,
// 256: 16.19) and config 4 (64: 2.36 ms, 32: 2.39).  lb_set_option(LB_OPT_ZC) overrides.
// k_step_node (with the CTA count padded to whole waves, tma_grid) is faster on shorter chunks than the model says: 512^3 64 planes
// 15.42 ms, 128: 15.79, 32: 15.76, 256: 16.04; 256^3 64 / 32: 1.97, 128: 2.02 (k_step_tma: 512^3 128: 15.70, 64: 15.80; fp32 128: 9.25,
// 64: 9.36): for it the candidates are the divisors of nz between 16 and 64, when there are any.
int effective_kernel(const lb_ctx* c);
int tma_zc(const lb_ctx* c) {
    if (c->zc_req >= 1) {                                             // the kernel wants whole chunks: the largest divisor of nz <= the request
        int zc = c->zc_req < c->nz ? c->zc_req : c->nz;
        while (c->nz % zc != 0) --zc;
        return zc;
    }
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    const double tiles = double(c->nx / OP_TX) * (c->ny / OP_TY);
    const double a = 0.5;
    int best = c->nz;
    double best_cost = 1e300;
    bool short_only = false;
    if (effective_kernel(c) == LB_KERNEL_NODE && tiles * c->nz / 64.0 >= 2.0 * sms)      // (small boxes: the model below)
        for (int zc = 16; zc <= 64 && zc <= c->nz; ++zc) short_only = short_only || c->nz % zc == 0;
    for (int zc = 1; zc <= c->nz; ++zc) {
        if (c->nz % zc != 0 || (short_only && (zc < 16 || zc > 64))) continue;
        const double waves = tiles * (c->nz / zc) / sms;
        const double cost = (zc + 4.0) * ((waves > 1.0 ? waves : 1.0) + a);
        if (cost < best_cost) { best_cost = cost; best = zc; }
    }
    return best;
}

// LB_KERNEL_HALO has no bounce-back: a box with solid nodes runs the TMA kernel instead (decided per step, effective_kernel)
int resolve_kernel(lb_ctx* c, int kind) {
    const bool tma_ok = onepass_ok(c) && c->have_tmap;
    if (kind == LB_KERNEL_AUTO) return tma_ok ? LB_KERNEL_TMA : (onepass_ok(c) ? LB_KERNEL_ONEPASS : LB_KERNEL_TWOPASS);
    if (kind == LB_KERNEL_ONEPASS && !onepass_ok(c)) return -1;
    if ((kind == LB_KERNEL_TMA || kind == LB_KERNEL_HALO || kind == LB_KERNEL_NODE) && !tma_ok) return -1;
    return kind;
}

// The later operators run k_collide_next on the two-pass path, except the colour gradient on a box without solids whose kernel
// choice resolves to a TMA-staged kernel: k_step_tma and k_step_node have their own variants of it.
bool next_path(const lb_ctx* c) {
    if (c->nsph > 0) return true;
    if (c->model == LB_MODEL_SHAN_CHEN) return false;
    return c->has_solid || (c->kernel != LB_KERNEL_TMA && c->kernel != LB_KERNEL_NODE);
}
int effective_kernel(const lb_ctx* c) {
    if (next_path(c)) return LB_KERNEL_TWOPASS;                                      // the later operators: general two-pass path
    if ((c->kernel == LB_KERNEL_HALO || c->kernel == LB_KERNEL_NODE) && c->has_solid) return LB_KERNEL_TMA;
    // Left to itself (AUTO) a plain fp64 Shan-Chen box runs the one-thread-per-node mapping of the TMA kernel: a third fewer
    // instructions for the same bytes, which under the board's power cap is worth 0.3 % over 20 steps and 1.1 % over 200 at 512^3
    // (fp32: the (node, component) mapping is 2 % faster).
    // The colour gradient gains most from it (one colour-blind collision per node instead of one per component): 256^3 fp64 2.32 ->
    // 2.01 ms, 512^3 17.9 -> 16.3; fp32 the same to 1 % either way.
    if (c->kernel == LB_KERNEL_TMA && c->kernel_req == LB_KERNEL_AUTO && c->dtype == LB_F64 && !c->has_solid)
        return LB_KERNEL_NODE;
    return c->kernel;
}

long long round64(long long v) { return (v + 63) / 64 * 64; }

}  // namespace

// the library's error slot (one per thread), shared with lb_single.cu
void lb_set_error(int code, const char* what) { g_err = what; g_err_code = code; }

// With a kernel that carries the density from step to step (TMA, one-pass) the planes travel WITH their carried density (rho_in
// and the three edge arrays, all z-major per component): the receiver's ghost planes then hold what the owner computed, the
// carried density stays valid and the one-pass kernels keep running on slabs.  Other kernels: populations only.
static bool planes_carry_density(const lb_ctx* c) {
    const int k = effective_kernel(c);
    return (k == LB_KERNEL_TMA || k == LB_KERNEL_NODE || k == LB_KERNEL_ONEPASS) && c->rho_x[0] != nullptr;
}
static size_t plane_buffer_elems(const lb_ctx* c, int nplanes) {
    const size_t pl = size_t(c->nx) * c->ny;
    size_t n = size_t(NPOP) * nplanes * pl;
    if (planes_carry_density(c)) {
        const size_t ntx = c->nx / OP_TX, nty = c->ny / OP_TY;
        n += size_t(2) * nplanes * (pl + nty * ntx * 2 * OP_TY + nty * 2 * c->nx + nty * ntx * 4);
    }
    return n;
}
template <typename T>
static int plane_copy_t(lb_ctx* c, int z0, int nplanes, T* dev, bool out) {
    const size_t pl = size_t(c->nx) * c->ny;
    auto copy = [&](T* buf, T* arr, size_t comp_stride, size_t per_z, int rows) -> cudaError_t {
        const size_t width = size_t(nplanes) * per_z * sizeof(T);
        T* state = arr + size_t(z0) * per_z;
        return out ? cudaMemcpy2DAsync(buf, width, state, comp_stride * sizeof(T), width, rows, cudaMemcpyDeviceToDevice, c->stream)
                   : cudaMemcpy2DAsync(state, comp_stride * sizeof(T), buf, width, width, rows, cudaMemcpyDeviceToDevice, c->stream);
    };
    const bool dens = planes_carry_density(c);
    if (dens && out) {                           // what leaves must describe the state
        const int rc = ensure_rho<T>(c);
        if (rc != LB_OK) return rc;
    }
    T* buf = dev;
    CU(copy(buf, static_cast<T*>(c->f[c->cur]), size_t(c->NP), pl, NPOP));
    buf += size_t(NPOP) * nplanes * pl;
    if (dens) {
        const size_t ntx = c->nx / OP_TX, nty = c->ny / OP_TY;
        const size_t psx = nty * ntx * 2 * OP_TY, psy = nty * 2 * size_t(c->nx), psxy = nty * ntx * 4;
        const int r = c->rcur;
        CU(copy(buf, static_cast<T*>(c->rho_in[r]), size_t(c->NP), pl, 2));    buf += size_t(2) * nplanes * pl;
        CU(copy(buf, static_cast<T*>(c->rho_x[r]), size_t(c->s_x), psx, 2));   buf += size_t(2) * nplanes * psx;
        CU(copy(buf, static_cast<T*>(c->rho_y[r]), size_t(c->s_y), psy, 2));   buf += size_t(2) * nplanes * psy;
        CU(copy(buf, static_cast<T*>(c->rho_xy[r]), size_t(c->s_xy), psxy, 2));
    }
    if (!out) {
        if (!dens) c->rho_valid = false;         // the carried density no longer describes the state
        c->hx_valid = false;                     // nor do the x-halo copies and the fused sums
        c->diag_fresh = false;
    }
    return LB_OK;
}
static int plane_copy(lb_ctx* c, int z0, int nplanes, void* dev, bool out) {
    if (!c || !dev) return fail(LB_EINVAL, "NULL argument");
    if (z0 < 0 || nplanes < 1 || z0 + nplanes > c->nz) return fail(LB_EINVAL, "plane range outside the box (no wrap)");
    if (!c->have_fields) return fail(LB_ESTATE, "no state to exchange yet");
    DeviceGuard guard(c->device);
    return c->dtype == LB_F64 ? plane_copy_t<double>(c, z0, nplanes, static_cast<double*>(dev), out)
                              : plane_copy_t<float>(c, z0, nplanes, static_cast<float*>(dev), out);
}

// ----------------------------------------------------------------------------------------
// C ABI
// ----------------------------------------------------------------------------------------
extern "C" {

const char* lb_last_error(void) { return g_err.c_str(); }
int lb_last_error_code(void) { return g_err_code; }
const char* lb_version(void) { return "lb-b200 0.2 (sm_100a)"; }

lb_ctx* lb_create_ex(int nx, int ny, int nz, double tau_r, double tau_b, double G, int dtype, void* cuda_stream) {
    g_err.clear();
    g_err_code = LB_OK;
    if (nx < 1 || ny < 1 || nz < 1) { fail(LB_EINVAL, "box dimensions must be >= 1"); return nullptr; }
    if ((long long)nx * ny * nz > (1ll << 31) - 1) { fail(LB_EINVAL, "box too large (N must fit in 31 bits)"); return nullptr; }
    if (ny > 65535 || nz > 65535) { fail(LB_EINVAL, "ny and nz must be <= 65535 (one thread block row per (y, z))"); return nullptr; }
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
    e = cudaGetDevice(&c->device);
    if (e != cudaSuccess) { fail_cuda(e, "cudaGetDevice"); delete c; return nullptr; }
    c->nx = nx; c->ny = ny; c->nz = nz;
    c->N = (long long)nx * ny * nz;
    c->NP = round64(c->N);
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
    for (int r = 0; r < 2; ++r) ok = ok && cudaMalloc(&c->rho_in[r], size_t(2) * c->NP * es) == cudaSuccess;
    if (onepass_ok(c)) {
        const long long ntx = nx / OP_TX, nty = ny / OP_TY;
        c->s_x = round64((long long)nz * nty * ntx * 2 * OP_TY);
        c->s_y = round64((long long)nz * nty * 2 * nx);
        c->s_xy = round64((long long)nz * nty * ntx * 4);
        for (int r = 0; r < 2; ++r) {
            ok = ok && cudaMalloc(&c->rho_x[r], size_t(2) * c->s_x * es) == cudaSuccess;
            ok = ok && cudaMalloc(&c->rho_y[r], size_t(2) * c->s_y * es) == cudaSuccess;
            ok = ok && cudaMalloc(&c->rho_xy[r], size_t(2) * c->s_xy * es) == cudaSuccess;
            ok = ok && cudaMalloc(&c->rho_er[r], size_t(2) * c->s_y * es) == cudaSuccess;
            ok = ok && cudaMalloc(&c->rho_ec[r], size_t(2) * c->s_x * es) == cudaSuccess;
        }
        c->hx_elems = (long long)2 * NHALO * nz * ntx * ny;
        for (int b = 0; b < 2; ++b) ok = ok && cudaMalloc(&c->hx[b], size_t(c->hx_elems) * es) == cudaSuccess;
    }
    ok = ok && cudaMalloc(&c->links, size_t(c->N) * sizeof(unsigned)) == cudaSuccess;
    c->stage_nodes = c->N < STAGE_NODES ? c->N : STAGE_NODES;
    ok = ok && cudaMalloc(&c->stage, size_t(c->stage_nodes) * 5 * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->diag_part, size_t(DIAG_BLOCKS) * 5 * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&c->diag_out, 5 * sizeof(double)) == cudaSuccess;
    if (ok) {
        ok = ok && cudaMemsetAsync(c->f[0], 0, fbytes, c->stream) == cudaSuccess;
        ok = ok && cudaMemsetAsync(c->f[1], 0, fbytes, c->stream) == cudaSuccess;
        ok = ok && cudaMemsetAsync(c->links, 0, size_t(c->N) * sizeof(unsigned), c->stream) == cudaSuccess;
    }
    if (!ok) {
        e = cudaGetLastError();
        lb_destroy(c);
        fail_cuda(e, "device allocation failed");        // LB_ENOMEM for an out-of-memory, LB_ECUDA otherwise
        return nullptr;
    }
    if (onepass_ok(c) && (dtype == LB_F64 ? configure_onepass_kernels<double>() : configure_onepass_kernels<float>()) != LB_OK) {
        lb_destroy(c);
        return nullptr;                                  // LB_ECUDA, message set
    }
    c->have_tmap = onepass_ok(c) && make_tmaps(c);
    c->balance = true;
    c->na_scratch = noalloc_scratch_address(c->device);  // set-up for lb_diagnostics_noalloc; a failure is reported there
    c->kernel_req = LB_KERNEL_AUTO;
    c->kernel = resolve_kernel(c, LB_KERNEL_AUTO);
    c->zc = onepass_zc(c);
    c->zc_tma = tma_zc(c);
    return c;
}

lb_ctx* lb_create(int nx, int ny, int nz, double tau_r, double tau_b, double G) {
    return lb_create_ex(nx, ny, nz, tau_r, tau_b, G, LB_F64, nullptr);
}

void lb_destroy(lb_ctx* c) {
    if (!c) return;
    DeviceGuard guard(c->device);
    cudaStreamSynchronize(c->stream);
    cudaFree(c->f[0]); cudaFree(c->f[1]); cudaFree(c->links);
    for (int r = 0; r < 2; ++r) {
        cudaFree(c->rho_in[r]); cudaFree(c->rho_x[r]); cudaFree(c->rho_y[r]); cudaFree(c->rho_xy[r]);
        cudaFree(c->rho_er[r]); cudaFree(c->rho_ec[r]); cudaFree(c->hx[r]);
    }
    cudaFree(c->stage); cudaFree(c->diag_part); cudaFree(c->diag_out); cudaFree(c->diag_cta);
    cudaFree(c->sph); cudaFree(c->pid);
    if (c->own_stream) cudaStreamDestroy(c->stream);
    delete c;
}

int lb_sync(lb_ctx* c) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    DeviceGuard guard(c->device);
    CU(cudaStreamSynchronize(c->stream));
    return LB_OK;
}

long long lb_launch_count(const lb_ctx* c) { return c ? c->launches : 0; }

int lb_get_kernel(const lb_ctx* c) { return c ? effective_kernel(c) : -1; }

int lb_set_option(lb_ctx* c, int option, long long value) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    DeviceGuard guard(c->device);
    switch (option) {
    case LB_OPT_ZC:
        if (value < 0 || value > c->nz) return fail(LB_EINVAL, "LB_OPT_ZC: 0 (heuristic) or 1..nz planes per CTA");
        c->zc_req = int(value);
        c->zc = onepass_zc(c);
        c->zc_tma = tma_zc(c);
        return LB_OK;
    case LB_OPT_DIAG:
        if (value != 0 && value != 1) return fail(LB_EINVAL, "LB_OPT_DIAG: 0 or 1");
        c->diag_mode = int(value);
        c->diag_fresh = false;
        return LB_OK;
    case LB_OPT_BALANCE:
        if (value != 0 && value != 1) return fail(LB_EINVAL, "LB_OPT_BALANCE: 0 or 1");
        c->balance = value != 0;
        return LB_OK;
    default:
        return fail(LB_EINVAL, "unknown option");
    }
}

long long lb_get_option(const lb_ctx* c, int option) {
    if (!c) return -1;
    switch (option) {
    case LB_OPT_ZC: return (c->kernel == LB_KERNEL_TMA || c->kernel == LB_KERNEL_HALO || c->kernel == LB_KERNEL_NODE) ? tma_zc(c) : c->zc;
    case LB_OPT_DIAG: return c->diag_mode;
    case LB_OPT_BALANCE: return c->balance ? 1 : 0;
    default: return -1;
    }
}

int lb_set_kernel(lb_ctx* c, int kind) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    if (kind != LB_KERNEL_AUTO && kind != LB_KERNEL_TWOPASS && kind != LB_KERNEL_ONEPASS && kind != LB_KERNEL_TMA && kind != LB_KERNEL_HALO &&
        kind != LB_KERNEL_NODE)
        return fail(LB_EINVAL, "unknown kernel kind");
    const int r = resolve_kernel(c, kind);
    if (r < 0) return fail(LB_EINVAL, "box shape does not allow this kernel");
    if (r != c->kernel) c->rho_valid = false;               // the density edge arrays are laid out per tile shape
    c->kernel_req = kind;
    c->kernel = r;
    return LB_OK;
}

int lb_set_solid_mask(lb_ctx* c, const unsigned char* mask) {
    if (!c || !mask) return fail(LB_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    const bool f64 = c->dtype == LB_F64;
    int rc;
    // the fields already set are defined on nodes (f): take them out of the h-state under the OLD links
    if (c->have_fields) {
        rc = f64 ? stream_to_scratch<double>(c) : stream_to_scratch<float>(c);
        if (rc != LB_OK) return rc;
    }
    bool any_solid = false;
    for (long long n = 0; n < c->N && !any_solid; ++n) any_solid = mask[n] != 0;
    // the mask travels through the staging buffer when it fits there, else through a temporary
    const bool own_tmp = size_t(c->N) > size_t(c->stage_nodes) * 5 * sizeof(double);
    unsigned char* d_mask = reinterpret_cast<unsigned char*>(c->stage);
    if (own_tmp) CU(cudaMalloc(&d_mask, size_t(c->N)));
    cudaError_t e = cudaMemcpyAsync(d_mask, mask, size_t(c->N), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) {
        k_build_links<<<blocks_for(c->N, 256), 256, 0, c->stream>>>(d_mask, c->links, c->nx, c->ny, c->nz);
        c->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (own_tmp) cudaFree(d_mask);
    if (e != cudaSuccess) return fail_cuda(e, "lb_set_solid_mask");
    c->has_solid = any_solid;   // a mask without solid nodes keeps the plain (no link word) kernels
    c->zc_tma = tma_zc(c);      // the chunk length that balances best depends on it
    if (!c->in_set_spheres) c->nsph = 0;   // a plain mask: every solid at rest
    c->rho_valid = false;
    if (!any_solid) {
        if (c->have_fields) return c->dtype == LB_F64 ? unstream_scratch<double>(c) : unstream_scratch<float>(c);
        return LB_OK;
    }
    // S8: solid nodes hold exactly 0 in both buffers (the step kernels never write them)
    rc = f64 ? zero_solids<double>(c, c->cur ^ 1) : zero_solids<float>(c, c->cur ^ 1);
    if (rc != LB_OK) return rc;
    if (c->have_fields) return f64 ? unstream_scratch<double>(c) : unstream_scratch<float>(c);
    return f64 ? zero_solids<double>(c, c->cur) : zero_solids<float>(c, c->cur);
}

int lb_set_colour_gradient(lb_ctx* c, double sigma, double beta) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    if (!std::isfinite(sigma) || !std::isfinite(beta) || beta < 0.0 || beta > 1.0) return fail(LB_EINVAL, "sigma must be finite, beta in [0, 1]");
    c->model = LB_MODEL_COLOUR_GRADIENT; c->sigma = sigma; c->beta = beta;
    c->rho_valid = false;
    return LB_OK;
}

int lb_set_shan_chen(lb_ctx* c) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    c->model = LB_MODEL_SHAN_CHEN;
    c->rho_valid = false;
    return LB_OK;
}

int lb_set_spheres(lb_ctx* c, int np, const double* centres, double radius, const double* vel, const double* omega) {
    if (!c || np < 0 || (np > 0 && (!centres || !(radius > 0.0)))) return fail(LB_EINVAL, "lb_set_spheres: bad arguments");
    DeviceGuard guard(c->device);
    // solid mask (reading S9) and the sphere of every solid node: integer work on the host, one pass over the spheres' bounding boxes
    std::string mask;
    int* pid = nullptr;
    try { mask.assign(size_t(c->N), char(0)); pid = new int[size_t(c->N)]; } catch (...) { return fail(LB_ENOMEM, "host allocation failed"); }
    for (long long n = 0; n < c->N; ++n) pid[n] = -1;
    const int reach = int(std::floor(radius)) + 1;
    const int dim[3] = {c->nx, c->ny, c->nz};
    for (int p = 0; p < np; ++p) {
        const double* ce = centres + 3 * p;
        int lo[3], hi[3];
        for (int a = 0; a < 3; ++a) { lo[a] = int(std::floor(ce[a])) - reach; hi[a] = int(std::floor(ce[a])) + reach + 1; }
        for (int a = 0; a < 3; ++a) if (hi[a] - lo[a] + 1 > dim[a]) { lo[a] = 0; hi[a] = dim[a] - 1; }
        for (int z = lo[2]; z <= hi[2]; ++z)
            for (int y = lo[1]; y <= hi[1]; ++y)
                for (int x = lo[0]; x <= hi[0]; ++x) {
                    const int q[3] = {((x % dim[0]) + dim[0]) % dim[0], ((y % dim[1]) + dim[1]) % dim[1], ((z % dim[2]) + dim[2]) % dim[2]};
                    double d2 = 0.0;
                    for (int a = 0; a < 3; ++a) {
                        double d = std::fabs(q[a] - ce[a]);
                        d = std::fmin(d, dim[a] - d);
                        d2 += d * d;
                    }
                    const long long n = q[0] + (long long)dim[0] * (q[1] + (long long)dim[1] * q[2]);
                    if (d2 <= radius * radius && pid[n] < 0) { mask[size_t(n)] = 1; pid[n] = p; }
                }
    }
    cudaFree(c->sph); cudaFree(c->pid);
    c->sph = nullptr; c->pid = nullptr;
    int rc = LB_OK;
    if (np > 0) {
        cudaError_t e = cudaMalloc(&c->sph, size_t(15) * np * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc(&c->pid, size_t(c->N) * sizeof(int));
        if (e == cudaSuccess) e = cudaMemsetAsync(c->sph, 0, size_t(15) * np * sizeof(double), c->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(c->sph, centres, size_t(3) * np * sizeof(double), cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess && vel) e = cudaMemcpyAsync(c->sph + 3 * np, vel, size_t(3) * np * sizeof(double), cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess && omega) e = cudaMemcpyAsync(c->sph + 6 * np, omega, size_t(3) * np * sizeof(double), cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(c->pid, pid, size_t(c->N) * sizeof(int), cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) rc = fail_cuda(e, "lb_set_spheres");
    }
    delete[] pid;
    if (rc != LB_OK) return rc;
    c->in_set_spheres = true;
    rc = lb_set_solid_mask(c, reinterpret_cast<const unsigned char*>(mask.data()));
    c->in_set_spheres = false;
    if (rc != LB_OK) return rc;
    c->nsph = np; c->radius = radius;
    return LB_OK;
}

// ---- slab decomposition: whole z planes of the device state to / from a caller-owned DEVICE buffer ----
int lb_export_planes(lb_ctx* c, int z0, int nplanes, void* device_dst) { return plane_copy(c, z0, nplanes, device_dst, true); }
int lb_import_planes(lb_ctx* c, int z0, int nplanes, const void* device_src) { return plane_copy(c, z0, nplanes, const_cast<void*>(device_src), false); }
long long lb_plane_buffer_bytes(const lb_ctx* c, int nplanes) {
    if (!c || nplanes < 1) return -1;
    return (long long)(plane_buffer_elems(c, nplanes) * esize(c));
}

int lb_get_sphere_forces(lb_ctx* c, double* F, double* T) {
    if (!c || !F || !T) return fail(LB_EINVAL, "NULL argument");
    if (c->nsph == 0) return LB_OK;
    DeviceGuard guard(c->device);
    CU(cudaMemcpyAsync(F, c->sph + 9 * c->nsph, size_t(3) * c->nsph * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaMemcpyAsync(T, c->sph + 12 * c->nsph, size_t(3) * c->nsph * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return LB_OK;
}

int lb_set_fields(lb_ctx* c, const double* rho_r, const double* rho_b, const double* ux, const double* uy, const double* uz) {
    if (!c || !rho_r || !rho_b) return fail(LB_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    const int nu = (ux != nullptr) + (uy != nullptr) + (uz != nullptr);
    if (nu != 0 && nu != 3) return fail(LB_EINVAL, "ux, uy, uz must be all NULL or all non-NULL");
    const double* src[5] = {rho_r, rho_b, ux, uy, uz};
    void* scratch = c->f[c->cur ^ 1];
    for (long long n0 = 0; n0 < c->N; n0 += c->stage_nodes) {
        const long long cnt = (c->N - n0 < c->stage_nodes) ? c->N - n0 : c->stage_nodes;
        double* st[5];
        for (int a = 0; a < 5; ++a) {
            st[a] = src[a] ? c->stage + a * c->stage_nodes : nullptr;
            if (src[a]) CU(cudaMemcpyAsync(st[a], src[a] + n0, size_t(cnt) * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        }
        const unsigned* lk = c->has_solid ? c->links : nullptr;
        if (c->dtype == LB_F64)
            k_init_eq<double><<<blocks_for(cnt, 128), 128, 0, c->stream>>>(static_cast<double*>(scratch), c->NP, n0, cnt, st[0], st[1], st[2], st[3], st[4], lk);
        else
            k_init_eq<float><<<blocks_for(cnt, 128), 128, 0, c->stream>>>(static_cast<float*>(scratch), c->NP, n0, cnt, st[0], st[1], st[2], st[3], st[4], lk);
        c->launches++;
        CU(cudaGetLastError());
    }
    const int rc = c->dtype == LB_F64 ? unstream_scratch<double>(c) : unstream_scratch<float>(c);
    if (rc != LB_OK) return rc;
    CU(cudaStreamSynchronize(c->stream));          // the caller's arrays are free again
    c->have_fields = true;
    return LB_OK;
}

int lb_set_populations(lb_ctx* c, const double* f) {
    if (!c || !f) return fail(LB_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    void* scratch = c->f[c->cur ^ 1];
    for (int q = 0; q < NPOP; ++q) {                    // ABI order [k][i] -> plane pop_plane(k, i)
        const double* src = f + (long long)q * c->N;
        const long long pq = pop_plane(q / Q, q % Q);
        if (c->dtype == LB_F64) {
            CU(cudaMemcpyAsync(static_cast<double*>(scratch) + pq * c->NP, src, size_t(c->N) * 8, cudaMemcpyHostToDevice, c->stream));
        } else {
            float* dst = static_cast<float*>(scratch) + pq * c->NP;
            for (long long n0 = 0; n0 < c->N; n0 += c->stage_nodes * 5) {
                const long long cnt = (c->N - n0 < c->stage_nodes * 5) ? c->N - n0 : c->stage_nodes * 5;
                CU(cudaMemcpyAsync(c->stage, src + n0, size_t(cnt) * 8, cudaMemcpyHostToDevice, c->stream));
                k_from_double<float><<<blocks_for(cnt, 256), 256, 0, c->stream>>>(c->stage, dst + n0, cnt);
                c->launches++;
                CU(cudaGetLastError());
            }
        }
    }
    int rc;
    if (c->has_solid) {
        rc = c->dtype == LB_F64 ? zero_solids<double>(c, c->cur ^ 1) : zero_solids<float>(c, c->cur ^ 1);
        if (rc != LB_OK) return rc;
    }
    rc = c->dtype == LB_F64 ? unstream_scratch<double>(c) : unstream_scratch<float>(c);
    if (rc != LB_OK) return rc;
    CU(cudaStreamSynchronize(c->stream));
    c->have_fields = true;
    return LB_OK;
}

int lb_step(lb_ctx* c, int nsteps) {
    if (!c) return fail(LB_EINVAL, "NULL context");
    DeviceGuard guard(c->device);
    if (nsteps < 0) return fail(LB_EINVAL, "nsteps must be >= 0");
    if (!c->have_fields) return fail(LB_ESTATE, "lb_step before lb_set_fields / lb_set_populations");
    c->zc_tma = tma_zc(c);                    // depends on which kernel the state of the context selects
    for (int s = 0; s < nsteps; ++s) {
        int rc;
        const int kern = effective_kernel(c);
        if (next_path(c)) rc = c->dtype == LB_F64 ? step_next<double>(c) : step_next<float>(c);
        else if (kern == LB_KERNEL_HALO) rc = c->dtype == LB_F64 ? step_halo<double>(c) : step_halo<float>(c);
        else if (kern == LB_KERNEL_NODE) rc = c->dtype == LB_F64 ? step_node<double>(c) : step_node<float>(c);
        else if (kern == LB_KERNEL_TMA) rc = c->dtype == LB_F64 ? step_tma<double>(c) : step_tma<float>(c);
        else if (kern == LB_KERNEL_ONEPASS) rc = c->dtype == LB_F64 ? step_onepass<double>(c) : step_onepass<float>(c);
        else rc = c->dtype == LB_F64 ? step_twopass<double>(c) : step_twopass<float>(c);
        if (rc != LB_OK) return rc;
    }
    return LB_OK;
}

int lb_get_populations(lb_ctx* c, double* f) {
    if (!c || !f) return fail(LB_EINVAL, "NULL argument");
    DeviceGuard guard(c->device);
    const int rc = c->dtype == LB_F64 ? stream_to_scratch<double>(c) : stream_to_scratch<float>(c);
    if (rc != LB_OK) return rc;
    const void* scratch = c->f[c->cur ^ 1];
    for (int q = 0; q < NPOP; ++q) {                    // plane pop_plane(k, i) -> ABI order [k][i]
        double* dst = f + (long long)q * c->N;
        const long long pq = pop_plane(q / Q, q % Q);
        if (c->dtype == LB_F64) {
            CU(cudaMemcpyAsync(dst, static_cast<const double*>(scratch) + pq * c->NP, size_t(c->N) * 8, cudaMemcpyDeviceToHost, c->stream));
        } else {
            const float* src = static_cast<const float*>(scratch) + pq * c->NP;
            for (long long n0 = 0; n0 < c->N; n0 += c->stage_nodes * 5) {
                const long long cnt = (c->N - n0 < c->stage_nodes * 5) ? c->N - n0 : c->stage_nodes * 5;
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
    DeviceGuard guard(c->device);
    double* dst[5] = {rho_r, rho_b, ux, uy, uz};
    const unsigned* lk = c->has_solid ? c->links : nullptr;
    for (long long n0 = 0; n0 < c->N; n0 += c->stage_nodes) {
        const long long cnt = (c->N - n0 < c->stage_nodes) ? c->N - n0 : c->stage_nodes;
        double* st[5];
        for (int a = 0; a < 5; ++a) st[a] = c->stage + a * c->stage_nodes;
        if (c->dtype == LB_F64)
            k_moments_out<double><<<blocks_for(cnt, 128), 128, 0, c->stream>>>(static_cast<const double*>(c->f[c->cur]), lk, c->NP, c->nx, c->ny, c->nz, n0, cnt, st[0], st[1], st[2], st[3], st[4]);
        else
            k_moments_out<float><<<blocks_for(cnt, 128), 128, 0, c->stream>>>(static_cast<const float*>(c->f[c->cur]), lk, c->NP, c->nx, c->ny, c->nz, n0, cnt, st[0], st[1], st[2], st[3], st[4]);
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
    DeviceGuard guard(c->device);
    unsigned* st = reinterpret_cast<unsigned*>(c->stage);
    const long long chunk = c->stage_nodes * 10;          // staging holds 5*c->stage_nodes doubles
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
    DeviceGuard guard(c->device);
    const unsigned* lk = c->has_solid ? c->links : nullptr;
    if (c->diag_mode && c->diag_fresh) {
        // the last step (halo kernel, LB_OPT_DIAG) left the per-CTA sums of the current state behind: no population pass
        k_diag_final<<<1, 256, 0, c->stream>>>(c->diag_cta, int(c->diag_ncta), c->diag_out);
        c->launches += 1;
    } else {
    if (c->dtype == LB_F64)
        k_diag_partial<double><<<DIAG_BLOCKS, 256, 0, c->stream>>>(static_cast<const double*>(c->f[c->cur]), lk, c->NP, c->nx, c->ny, c->nz, c->diag_part);
    else
        k_diag_partial<float><<<DIAG_BLOCKS, 256, 0, c->stream>>>(static_cast<const float*>(c->f[c->cur]), lk, c->NP, c->nx, c->ny, c->nz, c->diag_part);
    k_diag_final<<<1, 256, 0, c->stream>>>(c->diag_part, DIAG_BLOCKS, c->diag_out);
    c->launches += 2;
    }
    CU(cudaGetLastError());
    double h[5];
    CU(cudaMemcpyAsync(h, c->diag_out, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    mass[0] = h[0]; mass[1] = h[1];
    momentum[0] = h[2]; momentum[1] = h[3]; momentum[2] = h[4];
    return LB_OK;
}

// see include/lb.h.  No cudaMalloc / cudaFree / memcpy / synchronisation: two launches on the context's stream.
int lb_diagnostics_noalloc(lb_ctx* c, double* out_dev) {
    if (!c || !out_dev) return fail(LB_EINVAL, "NULL argument");
    const long long nblocks = (c->N + NOALLOC_NODES_PER_BLOCK - 1) / NOALLOC_NODES_PER_BLOCK;
    if (nblocks > NOALLOC_MAX_BLOCKS)
        return fail(LB_EINVAL, "lb_diagnostics_noalloc: the box has more than 2^28 nodes, beyond the static scratch (16384 partials); use lb_get_diagnostics");
    if (!c->have_fields) return fail(LB_ESTATE, "lb_diagnostics_noalloc before lb_set_fields / lb_set_populations");
    if (!c->na_scratch) return fail(LB_ECUDA, "lb_diagnostics_noalloc: the address of the static scratch could not be obtained when the context was created");
    DeviceGuard guard(c->device);
    const unsigned* lk = c->has_solid ? c->links : nullptr;
    // every block overwrites its own partial and k_diag_final reads the first nblocks only: nothing has to start at zero,
    // whatever an earlier call (another context, another size) left in the array
    if (c->dtype == LB_F64)
        k_diag_partial<double><<<int(nblocks), 256, 0, c->stream>>>(static_cast<const double*>(c->f[c->cur]), lk, c->NP, c->nx, c->ny, c->nz, c->na_scratch);
    else
        k_diag_partial<float><<<int(nblocks), 256, 0, c->stream>>>(static_cast<const float*>(c->f[c->cur]), lk, c->NP, c->nx, c->ny, c->nz, c->na_scratch);
    k_diag_final<<<1, 256, 0, c->stream>>>(c->na_scratch, int(nblocks), out_dev);
    c->launches += 2;
    CU(cudaGetLastError());
    return LB_OK;
}

}  // extern "C"
