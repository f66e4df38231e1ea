// lb_oracle.cpp -- CPU ORACLE for the two-component Shan-Chen D3Q19 update.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
// It shares no code, header, table or helper with the CUDA path under
// paper_2112_08264_b200/csrc/ (not even the velocity table), and neither side
// includes or imports the other.
//
// Plain, slow, single-threaded, fp64.  No blocking, fusion or reordering beyond
// what the step-by-step statement below says, so that it can be checked against
// the paper by eye.  Build: g++ -O2 -ffp-contract=off (reference build).
//
// What it follows (PAPER.md = /root/reference/PAPER.md; SURVEY = SURVEY.md §8(c)):
//   * D3Q19 velocity set ............. PAPER.md:75 (§2); numbering = reading S1
//   * BGK update, Eq. 1 ............... PAPER.md:77-80
//   * two-component form, Eq. 5 ....... PAPER.md:314-318
//   * moments, Eq. 6-7 ................ PAPER.md:320-326
//   * equilibrium, Eq. 10, c_s^2=1/3 .. PAPER.md:338-342
//   * lattice weights 1/3,1/18,1/36 ... PAPER.md:393-398 (table)
//   * order collide -> bounce-back -> stream, PAPER.md:128-138 (§3)
//   * solid nodes skipped .............. PAPER.md:134
//   * halfway bounce-back, wall at rest, Eq. 23-24 with u_b = 0
//   * periodic box ..................... PAPER.md:160 (§5)
//   * one-step two-grid (old/new) ...... PAPER.md:124 (§3)
//   * Shan-Chen force, psi = rho, forcing scheme: the paper is silent; readings
//     S2-S8 of SURVEY §8(c) (listed in DESIGN.md §"Readings").
//
// Pins: every function here is pinned by tests/test_oracle_pins.py (P1-P12 of
// SURVEY §8(c)); none is "parity unpinned".
//
// One call ora_step does, with two full population buffers f (time t), g (t+1):
//
//   for every node x:                       # pass 1: densities
//       if solid(x): rho[k][x] = 0 for both k; continue
//       rho[k][x] = sum over i = 0..18, in index order, of f[k][i][x]
//   for every node x that is not solid:     # pass 2: force, collide, stream
//       j[k]   = sum_i f[k][i][x] * c_i
//       den    = om_r*rho[r][x] + om_b*rho[b][x],  om_k = 1/tau_k
//       u'     = (om_r*j[r] + om_b*j[b]) / den     (u' = 0 if den == 0)
//       for k in (r, b):
//           grad = sum over i = 1..18 of w_i * rho[kbar][(x+c_i) mod n] * c_i
//           du   = -G * grad               # = F^k/rho^k because psi = rho  (S2,S3,S6)
//           for i in 0..18:
//               fs = (1-om_k)*f[k][i][x] + om_k*feq_i(rho[k][x],u')
//                    + feq_i(rho[k][x],u'+du) - feq_i(rho[k][x],u')      (S5)
//               y  = (x + c_i) mod n
//               if solid(y): g[k][opp(i)][x] = fs     # halfway bounce-back
//               else:        g[k][i][y]      = fs     # stream
//   for every solid node x: g[k][i][x] = 0
//   swap f, g
//   feq_i(rho,u) = w_i*rho*(1 + 3 c_i.u + 4.5 (c_i.u)^2 - 1.5 u.u)
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>

namespace {

// Reading S1: direction numbering (part of the ABI, visible in get_populations).
const int CX[19] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
const int CY[19] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
const int CZ[19] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};

inline double weight(int i) {
    const int c2 = CX[i] * CX[i] + CY[i] * CY[i] + CZ[i] * CZ[i];
    return c2 == 0 ? 1.0 / 3.0 : (c2 == 1 ? 1.0 / 18.0 : 1.0 / 36.0);
}
inline int opp(int i) { return i == 0 ? 0 : ((i & 1) ? i + 1 : i - 1); }

// Eq. 10 with c_s^2 = 1/3.
inline double feq(int i, double rho, double ux, double uy, double uz) {
    const double cu = CX[i] * ux + CY[i] * uy + CZ[i] * uz;
    const double uu = ux * ux + uy * uy + uz * uz;
    return weight(i) * rho * (1.0 + 3.0 * cu + 4.5 * (cu * cu) - 1.5 * uu);
}

struct Ctx {
    int nx, ny, nz;
    size_t N;
    double tau[2], G;
    int forcing;                // 0 = exact-difference (default, S5), 1 = velocity shift
    bool have_fields;
    std::vector<double> f, g;   // [k][i][z][y][x]
    std::vector<double> rho;    // [k][n]
    std::vector<unsigned char> solid;
    size_t idx(int x, int y, int z) const { return (size_t)x + (size_t)nx * ((size_t)y + (size_t)ny * (size_t)z); }
    size_t nb(int x, int y, int z, int i) const {          // (x + c_i) mod n, any n >= 1 (S14)
        const int xn = ((x + CX[i]) % nx + nx) % nx;
        const int yn = ((y + CY[i]) % ny + ny) % ny;
        const int zn = ((z + CZ[i]) % nz + nz) % nz;
        return idx(xn, yn, zn);
    }
    double& F(std::vector<double>& a, int k, int i, size_t n) { return a[((size_t)k * 19 + i) * N + n]; }
};

// Neumaier compensated accumulation (diagnostics only).
struct Comp {
    double s = 0.0, c = 0.0;
    void add(double v) {
        const double t = s + v;
        if (std::fabs(s) >= std::fabs(v)) c += (s - t) + v; else c += (v - t) + s;
        s = t;
    }
    double value() const { return s + c; }
};

void zero_solids(Ctx* c, std::vector<double>& a) {
    for (size_t n = 0; n < c->N; ++n)
        if (c->solid[n])
            for (int k = 0; k < 2; ++k)
                for (int i = 0; i < 19; ++i) c->F(a, k, i, n) = 0.0;
}

void densities(Ctx* c) {                          // pass 1; Eq. 6
    for (size_t n = 0; n < c->N; ++n)
        for (int k = 0; k < 2; ++k) {
            double r = 0.0;
            if (!c->solid[n])
                for (int i = 0; i < 19; ++i) r += c->F(c->f, k, i, n);
            c->rho[(size_t)k * c->N + n] = r;
        }
}

// du^k = -G * sum_{i=1..18} w_i rho^{kbar}(x+c_i) c_i   (S2, S3, S6, S7)
void shan_chen_du(Ctx* c, int x, int y, int z, int k, double du[3]) {
    const int kb = 1 - k;
    double gx = 0.0, gy = 0.0, gz = 0.0;
    for (int i = 1; i < 19; ++i) {
        const double wr = weight(i) * c->rho[(size_t)kb * c->N + c->nb(x, y, z, i)];
        gx += wr * CX[i];
        gy += wr * CY[i];
        gz += wr * CZ[i];
    }
    du[0] = -c->G * gx;
    du[1] = -c->G * gy;
    du[2] = -c->G * gz;
}

void step_once(Ctx* c) {
    densities(c);
    const double om[2] = {1.0 / c->tau[0], 1.0 / c->tau[1]};
    for (int z = 0; z < c->nz; ++z)
        for (int y = 0; y < c->ny; ++y)
            for (int x = 0; x < c->nx; ++x) {
                const size_t n = c->idx(x, y, z);
                if (c->solid[n]) continue;
                double j[2][3];
                for (int k = 0; k < 2; ++k) {
                    j[k][0] = j[k][1] = j[k][2] = 0.0;
                    for (int i = 0; i < 19; ++i) {
                        const double v = c->F(c->f, k, i, n);
                        j[k][0] += v * CX[i];
                        j[k][1] += v * CY[i];
                        j[k][2] += v * CZ[i];
                    }
                }
                const double rr = c->rho[n], rb = c->rho[c->N + n];
                const double den = om[0] * rr + om[1] * rb;              // S4
                double u[3] = {0.0, 0.0, 0.0};
                if (den != 0.0)
                    for (int a = 0; a < 3; ++a) u[a] = (om[0] * j[0][a] + om[1] * j[1][a]) / den;
                for (int k = 0; k < 2; ++k) {
                    const double rk = c->rho[(size_t)k * c->N + n];
                    double du[3];
                    shan_chen_du(c, x, y, z, k, du);
                    for (int i = 0; i < 19; ++i) {
                        const double fi = c->F(c->f, k, i, n);
                        double fs;
                        if (c->forcing == 0) {
                            fs = (1.0 - om[k]) * fi + om[k] * feq(i, rk, u[0], u[1], u[2])
                                 + feq(i, rk, u[0] + du[0], u[1] + du[1], u[2] + du[2])
                                 - feq(i, rk, u[0], u[1], u[2]);
                        } else {            // alternative reading of S5: velocity shift
                            fs = (1.0 - om[k]) * fi
                                 + om[k] * feq(i, rk, u[0] + c->tau[k] * du[0], u[1] + c->tau[k] * du[1],
                                               u[2] + c->tau[k] * du[2]);
                        }
                        const size_t yb = c->nb(x, y, z, i);
                        if (c->solid[yb]) c->F(c->g, k, opp(i), n) = fs;   // Eq. 23-24, u_b = 0
                        else              c->F(c->g, k, i, yb) = fs;      // Eq. 1 / Eq. 5, streaming
                    }
                }
            }
    zero_solids(c, c->g);
    c->f.swap(c->g);
}

}  // namespace

extern "C" {

enum { ORA_OK = 0, ORA_EINVAL = -1, ORA_ENOMEM = -2, ORA_ESTATE = -4 };

void* ora_create(int nx, int ny, int nz, double tau_r, double tau_b, double G) {
    if (nx < 1 || ny < 1 || nz < 1) return nullptr;
    if (!(tau_r > 0.5) || !(tau_b > 0.5) || !std::isfinite(tau_r) || !std::isfinite(tau_b)) return nullptr;  // Eq. 2: 0 < omega < 2
    if (!std::isfinite(G)) return nullptr;
    Ctx* c = new (std::nothrow) Ctx();
    if (!c) return nullptr;
    c->nx = nx; c->ny = ny; c->nz = nz;
    c->N = (size_t)nx * ny * nz;
    c->tau[0] = tau_r; c->tau[1] = tau_b; c->G = G;
    c->forcing = 0;
    c->have_fields = false;
    try {
        c->f.assign(38 * c->N, 0.0);
        c->g.assign(38 * c->N, 0.0);
        c->rho.assign(2 * c->N, 0.0);
        c->solid.assign(c->N, 0);
    } catch (...) { delete c; return nullptr; }
    return c;
}

void ora_destroy(void* h) { delete static_cast<Ctx*>(h); }

int ora_set_forcing(void* h, int mode) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c || (mode != 0 && mode != 1)) return ORA_EINVAL;
    c->forcing = mode;
    return ORA_OK;
}

// f_i^k = f_i^eq(rho^k, u) at every node (Eq. 10); ux/uy/uz may be NULL (u = 0).
int ora_set_fields(void* h, const double* rho_r, const double* rho_b,
                   const double* ux, const double* uy, const double* uz) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c || !rho_r || !rho_b) return ORA_EINVAL;
    for (size_t n = 0; n < c->N; ++n) {
        const double u0 = ux ? ux[n] : 0.0, u1 = uy ? uy[n] : 0.0, u2 = uz ? uz[n] : 0.0;
        for (int i = 0; i < 19; ++i) {
            c->F(c->f, 0, i, n) = feq(i, rho_r[n], u0, u1, u2);
            c->F(c->f, 1, i, n) = feq(i, rho_b[n], u0, u1, u2);
        }
    }
    zero_solids(c, c->f);
    c->have_fields = true;
    return ORA_OK;
}

int ora_set_solid_mask(void* h, const unsigned char* mask) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c || !mask) return ORA_EINVAL;
    for (size_t n = 0; n < c->N; ++n) c->solid[n] = mask[n] ? 1 : 0;
    zero_solids(c, c->f);                                     // S8
    return ORA_OK;
}

int ora_set_populations(void* h, const double* f) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c || !f) return ORA_EINVAL;
    std::memcpy(c->f.data(), f, sizeof(double) * 38 * c->N);
    zero_solids(c, c->f);
    c->have_fields = true;
    return ORA_OK;
}

int ora_step(void* h, int nsteps) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c || nsteps < 0) return ORA_EINVAL;
    if (!c->have_fields) return ORA_ESTATE;
    for (int s = 0; s < nsteps; ++s) step_once(c);
    return ORA_OK;
}

int ora_get_populations(void* h, double* f) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c || !f) return ORA_EINVAL;
    std::memcpy(f, c->f.data(), sizeof(double) * 38 * c->N);
    return ORA_OK;
}

// rho^k (Eq. 6) and the barycentric velocity u = sum_k j^k / sum_k rho^k (Eq. 7).
int ora_get_moments(void* h, double* rho_r, double* rho_b, double* ux, double* uy, double* uz) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c) return ORA_EINVAL;
    densities(c);
    for (size_t n = 0; n < c->N; ++n) {
        double jx = 0.0, jy = 0.0, jz = 0.0;
        if (!c->solid[n])
            for (int k = 0; k < 2; ++k)
                for (int i = 0; i < 19; ++i) {
                    const double v = c->F(c->f, k, i, n);
                    jx += v * CX[i]; jy += v * CY[i]; jz += v * CZ[i];
                }
        const double r = c->rho[n] + c->rho[c->N + n];
        if (rho_r) rho_r[n] = c->rho[n];
        if (rho_b) rho_b[n] = c->rho[c->N + n];
        if (ux) ux[n] = r != 0.0 ? jx / r : 0.0;
        if (uy) uy[n] = r != 0.0 ? jy / r : 0.0;
        if (uz) uz[n] = r != 0.0 ? jz / r : 0.0;
    }
    return ORA_OK;
}

// bit i of links[n] set iff node n is fluid and (n + c_i) mod box is solid.
int ora_get_link_mask(void* h, unsigned int* links) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c || !links) return ORA_EINVAL;
    for (int z = 0; z < c->nz; ++z)
        for (int y = 0; y < c->ny; ++y)
            for (int x = 0; x < c->nx; ++x) {
                const size_t n = c->idx(x, y, z);
                unsigned int m = 0;
                if (!c->solid[n])
                    for (int i = 1; i < 19; ++i)
                        if (c->solid[c->nb(x, y, z, i)]) m |= 1u << i;
                links[n] = m;
            }
    return ORA_OK;
}

// mass[k] = sum_x rho^k, momentum = sum_x sum_k j^k over fluid nodes (compensated sums).
int ora_get_diagnostics(void* h, double mass[2], double momentum[3]) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c || !mass || !momentum) return ORA_EINVAL;
    Comp m[2], p[3];
    for (size_t n = 0; n < c->N; ++n) {
        if (c->solid[n]) continue;
        for (int k = 0; k < 2; ++k)
            for (int i = 0; i < 19; ++i) {
                const double v = c->F(c->f, k, i, n);
                m[k].add(v);
                if (CX[i]) p[0].add(v * CX[i]);
                if (CY[i]) p[1].add(v * CY[i]);
                if (CZ[i]) p[2].add(v * CZ[i]);
            }
    }
    mass[0] = m[0].value(); mass[1] = m[1].value();
    for (int a = 0; a < 3; ++a) momentum[a] = p[a].value();
    return ORA_OK;
}

// Shan-Chen force F^k(x) = rho^k(x) * du^k(x) of the current state, [a][n] with a = x,y,z.
int ora_get_force(void* h, double* F_r, double* F_b) {
    Ctx* c = static_cast<Ctx*>(h);
    if (!c || !F_r || !F_b) return ORA_EINVAL;
    densities(c);
    for (int z = 0; z < c->nz; ++z)
        for (int y = 0; y < c->ny; ++y)
            for (int x = 0; x < c->nx; ++x) {
                const size_t n = c->idx(x, y, z);
                for (int k = 0; k < 2; ++k) {
                    double du[3] = {0.0, 0.0, 0.0};
                    if (!c->solid[n]) shan_chen_du(c, x, y, z, k, du);
                    double* F = k == 0 ? F_r : F_b;
                    for (int a = 0; a < 3; ++a) F[(size_t)a * c->N + n] = c->rho[(size_t)k * c->N + n] * du[a];
                }
            }
    return ORA_OK;
}

// Eq. 10 for one (rho, u): out[19].
void ora_feq(double rho, double ux, double uy, double uz, double* out) {
    for (int i = 0; i < 19; ++i) out[i] = feq(i, rho, ux, uy, uz);
}

// The direction table as the oracle numbers it: c[19][3] (ints) and w[19].
void ora_lattice(int* c, double* w) {
    for (int i = 0; i < 19; ++i) {
        c[3 * i + 0] = CX[i]; c[3 * i + 1] = CY[i]; c[3 * i + 2] = CZ[i];
        w[i] = weight(i);
    }
}

}  // extern "C"
