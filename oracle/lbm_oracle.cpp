// ============================================================================
// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// A plain, slow, loop-based CPU implementation of the per-timestep Shan-Chen
// multiphase lattice-Boltzmann update of the JAX-LaB paper (arxiv 2506.17713),
// written from the paper (P:<line> = /root/reference/PAPER.md line) and the
// readings listed in DESIGN.md ("Readings", R1..R17; they restate SURVEY.md
// §8(c) G1..G17).  It follows the algorithm step by step, in the paper's
// order, over all cells with nested loops; sums run in index order i=0..q-1;
// there is no blocking, fusion or reordering (compile with -ffp-contract=off).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may load this library.  It shares no code, header, table or
// constant with paper_2506_17713_b200/csrc (the CUDA path).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"):
//   f_eq moments (closed form), mass/momentum conservation, pure streaming is
//   a permutation, MRT(S=I/tau) == BGK, EDM == shift at tau=1, EOS pressure ->
//   Maxwell densities of the paper's Table 1, psi=exp(-1/rho)
//   density ratio ~7.6, Laplace law, neutral wetting = 90 deg
//   (P:275), inlet mass flux rho_w*u_w per face cell, closed-box mass
//   conservation (halfway bounce-back).
//   viscosity nu = c_s^2 (tau - 1/2) from shear-wave decay, Poiseuille flow
//   between pressure faces (first-order pin of the anti-bounce-back faces).
//   A-weighted Zhang-Chen force (Eq. 11-13): F_ZC = -grad U against
//   a re-typed EOS, weighted sum, coexistence -> Maxwell with A ~ -0.19,
//   mass / momentum conservation.
//   Surface-tension control (Eq. 14-16, D2Q9 MRT): domain-summed moments after one
//   step = C of Eq. 15 with Q of Eq. 16 (incl. the A_kk term) evaluated by hand; sigma(kappa = 0.5)
//   / sigma(0) against the ratio of the paper's Table 2 (CS row: 0.457).
//   Single terms (tests/test_oracle_terms.py): velocity shift at tau != 1 and MRT (momentum gain per
//   step = total force, exactly), the w_i weights of rho_ave in Eq. 17 on a hand-built non-uniform
//   neighbourhood, Eq. 6's half force (u = (t + 1/2) a), D3Q19 MRT rate <-> row assignment (shear
//   waves on axes and face diagonals), and the O(u^2) bracket of the pressure face (a uniform
//   equilibrium flow at any Mach number is an exact fixed point between two pressure faces).
//   Contact angles of configs 2 and 4 (60 / 40 deg) from a circle fit of the meniscus.
//   PARITY UNPINNED: nothing on the step itself.  (Table 2's absolute surface tensions and the
//   Fig. 4-8 curves depend on unpublished alpha, A, kappa and are not reproduced.)
//
// State = post-stream populations f_i^k(x,t) (in the storage dtype, possibly
// shifted by w_i*rho_ref, reading R16).  One step = S1..S7 below.
// ============================================================================
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <string>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------- lattices
// Reading R1 (paper names the lattices only): the standard D2Q9 and
// D3Q19 velocity sets; order = rest, axis directions, diagonals.  The opposite
// table is derived by search, not typed.
const int E_D2Q9[9][3] = {
    {0, 0, 0},
    {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0},
    {1, 1, 0}, {-1, -1, 0}, {1, -1, 0}, {-1, 1, 0}};
const double W_D2Q9[9] = {4.0 / 9,
                          1.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9,
                          1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36};
const int E_D3Q19[19][3] = {
    {0, 0, 0},
    {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1},
    {1, 1, 0}, {-1, -1, 0}, {1, -1, 0}, {-1, 1, 0},
    {1, 0, 1}, {-1, 0, -1}, {1, 0, -1}, {-1, 0, 1},
    {0, 1, 1}, {0, -1, -1}, {0, 1, -1}, {0, -1, 1}};
const double W_D3Q19[19] = {1.0 / 3,
                            1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18, 1.0 / 18,
                            1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36,
                            1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36};

enum { LAT_D2Q9 = 0, LAT_D3Q19 = 1 };
enum { PSI_EOS_CS = 0, PSI_EOS_PR = 1, PSI_EOS_VDW = 2, PSI_EOS_RK = 3, PSI_EOS_RKS = 4,
       PSI_RHO = 5, PSI_EXP = 6, PSI_SC93 = 7 };
enum { COLL_BGK = 0, COLL_MRT = 1 };
enum { FORCE_EDM = 0, FORCE_SHIFT = 1 };
enum { DT_F16 = 0, DT_F32 = 1, DT_F64 = 2 };
enum { FACE_PERIODIC = 0, FACE_WALL = 1, FACE_VELOCITY = 2, FACE_PRESSURE = 3 };

}  // namespace

extern "C" {
// Plain-data configuration, mirrored field by field in oracle/lbm_oracle.py.
struct olbm_config {
    int32_t lattice;           // LAT_*
    int32_t nx, ny, nz;        // nz = 1 for D2Q9
    int32_t n_components;      // 1 or 2
    int32_t periodic[3];       // per axis
    int32_t psi_kind[2];       // PSI_*
    int32_t collision;         // COLL_*
    int32_t forcing;           // FORCE_*
    int32_t compute_dtype;     // DT_F32 / DT_F64
    int32_t store_dtype;       // DT_F16 / DT_F32 / DT_F64 (<= compute)
    int32_t no_collide;        // 1: f* = f (pure streaming test)
    double eos_a[2], eos_b[2], eos_R[2], eos_omega[2], eos_T[2];
    double alpha[2];           // pressure modification parameter alpha^k
    double rho0[2];            // SC93 psi = rho0 (1 - exp(-rho/rho0))
    double G[2][2];            // g_kk' of Eq. 13, weights w_i/c_s^2 (R2)
    double wet_phi[2], wet_drho[2], wet_lo[2], wet_hi[2];  // Eq. 17 + limiter
    double tau[2];             // BGK tau (MRT: the rates below decide; tau is not read)
    double mrt_rates[2][19];   // diagonal of S, moment order of R9
    double rho_ref;            // storage shift: stored = f_i - w_i*rho_ref (R16)
    double zc_A[2];            // A_kk of Eq. 11/13: F^k = A_kk F_ZC^k + (1 - A_kk) F_SC^k; 0 = pure Shan-Chen
    double body_accel[3];      // body force per unit mass a: F^k += rho^k a (reading R19)
    double st_kappa[2];        // kappa of Eq. 16: surface tension scales with 1 - kappa; D2Q9 + MRT only
};
}

namespace {

// -------------------------------------------------- equations of state (R3)
// The paper names the EOS but prints no formula; the textbook
// forms below with the Yuan & Schaefer parameters reproduce the Maxwell column
// of the paper's Table 1 -- tests/test_oracle_eos.py.
double eos_critical_temperature(int kind, double a, double b, double R) {
    switch (kind) {
        case PSI_EOS_CS:  return 0.3773 * a / (b * R);
        case PSI_EOS_PR:  return 0.0778 * a / (0.45724 * b * R);
        case PSI_EOS_VDW: return 8.0 * a / (27.0 * b * R);
        case PSI_EOS_RK:  return std::pow(0.08664 * a / (0.42748 * b * R), 2.0 / 3.0);
        case PSI_EOS_RKS: return 0.08664 * a / (0.42748 * b * R);
    }
    return 0.0;
}

template <class T>
T eos_pressure(int kind, T a, T b, T R, T omega, T Tabs, T Tc, T rho) {
    switch (kind) {
        case PSI_EOS_CS: {
            T eta = b * rho / T(4);
            T one_m = T(1) - eta;
            return rho * R * Tabs * (T(1) + eta + eta * eta - eta * eta * eta) / (one_m * one_m * one_m)
                   - a * rho * rho;
        }
        case PSI_EOS_PR: {
            T k = T(0.37464) + T(1.54226) * omega - T(0.26992) * omega * omega;
            T s = T(1) + k * (T(1) - std::sqrt(Tabs / Tc));
            T al = s * s;
            return rho * R * Tabs / (T(1) - b * rho)
                   - a * al * rho * rho / (T(1) + T(2) * b * rho - b * b * rho * rho);
        }
        case PSI_EOS_VDW:
            return rho * R * Tabs / (T(1) - b * rho) - a * rho * rho;
        case PSI_EOS_RK:
            return rho * R * Tabs / (T(1) - b * rho) - a * rho * rho / (std::sqrt(Tabs) * (T(1) + b * rho));
        case PSI_EOS_RKS: {
            T k = T(0.480) + T(1.574) * omega - T(0.176) * omega * omega;
            T s = T(1) + k * (T(1) - std::sqrt(Tabs / Tc));
            T al = s * s;
            return rho * R * Tabs / (T(1) - b * rho) - a * al * rho * rho / (T(1) + b * rho);
        }
    }
    return T(0);
}

// -------------------------------------------------- storage rounding (R16)
// fp16: round-to-nearest-even of a float to IEEE binary16, returned as float.
// Written on the bit pattern so it does not depend on compiler fp16 support.
float round_to_half(float v) {
    uint32_t x;
    std::memcpy(&x, &v, 4);
    uint32_t sign = x & 0x80000000u;
    uint32_t ax = x & 0x7fffffffu;
    float out;
    if (ax >= 0x7f800000u) {  // inf / nan
        return v;
    }
    if (ax >= 0x477ff000u) {  // >= 65520 rounds to inf
        uint32_t r = sign | 0x7f800000u;
        std::memcpy(&out, &r, 4);
        return out;
    }
    if (ax < 0x38800000u) {   // below the smallest normal half (2^-14): subnormal grid 2^-24
        float a;
        std::memcpy(&a, &ax, 4);
        // adding 2^-1 * 2^... : use the magic-number trick in float (exact RNE on the 2^-24 grid)
        const float magic = 0.5f;  // ulp(0.5f..1) = 2^-24 in float
        float r = (a + magic) - magic;
        uint32_t rb;
        std::memcpy(&rb, &r, 4);
        rb |= sign;
        std::memcpy(&out, &rb, 4);
        return out;
    }
    // normal half: keep 10 mantissa bits, RNE on the 13 dropped bits
    uint32_t lsb = (ax >> 13) & 1u;
    uint32_t r = ax + 0x0fffu + lsb;
    r &= ~0x1fffu;
    r |= sign;
    std::memcpy(&out, &r, 4);
    return out;
}

template <class T>
T round_store(T v, int store_dtype);
template <>
float round_store<float>(float v, int store_dtype) {
    return store_dtype == DT_F16 ? round_to_half(v) : v;
}
template <>
double round_store<double>(double v, int store_dtype) {
    if (store_dtype == DT_F32) return (double)(float)v;
    return v;  // DT_F64 (DT_F16 with fp64 compute is rejected at create)
}

// ---------------------------------------------------------------- simulator
struct SimBase {
    virtual ~SimBase() {}
    virtual int set_solid_mask(const uint8_t* m) = 0;
    virtual int set_face_bc(int face, int kind, const double* rho_w, const double* u_w) = 0;
    virtual int init_fields(const double* const* rho, const double* u) = 0;
    virtual int step(int n) = 0;
    virtual int get_macroscopic(double* const* rho, double* u, double* p) = 0;
    virtual int get_populations(int k, double* out) = 0;
    virtual int set_populations(int k, const double* in) = 0;
    virtual int get_link_flags(uint32_t* out) = 0;
    virtual int64_t get_boundary_solids(int64_t* out, int64_t cap) = 0;
    virtual int get_force(int k, double* out) = 0;
    virtual int get_psi(int k, double* out) = 0;
};

template <class T>
struct Sim : SimBase {
    olbm_config c;
    int d, q;
    const int (*e)[3];
    const double* w;
    int opp[19];
    int n[3];
    int64_t N;
    T cs2;
    T wT[19];        // lattice weights in T
    T gw[19];        // Green's function G(x,x+e_i) = w_i / c_s^2 (R2), in T
    T M[19][19], Minv[19][19];
    std::vector<uint8_t> solid;
    std::vector<int64_t> bsolid;  // solids with >= 1 fluid neighbour, ascending index (R11)
    int face_kind[6];
    double face_rho[6][2];
    double face_u[6][3];
    std::vector<T> f[2], fstar[2], rho[2], psi[2], U[2], j[2][3], F[2][3];
    std::vector<T> ucom[3];  // common velocity u' of S5
    int64_t steps_done = 0;

    explicit Sim(const olbm_config& cfg) : c(cfg) {
        if (c.lattice == LAT_D2Q9) { d = 2; q = 9; e = E_D2Q9; w = W_D2Q9; }
        else { d = 3; q = 19; e = E_D3Q19; w = W_D3Q19; }
        n[0] = c.nx; n[1] = c.ny; n[2] = c.nz;
        N = (int64_t)c.nx * c.ny * c.nz;
        cs2 = T(1) / T(3);
        for (int i = 0; i < q; ++i) {
            opp[i] = -1;
            for (int k = 0; k < q; ++k)
                if (e[k][0] == -e[i][0] && e[k][1] == -e[i][1] && e[k][2] == -e[i][2]) opp[i] = k;
            wT[i] = (T)w[i];
            gw[i] = (T)(w[i] * 3.0);
        }
        build_mrt();
        solid.assign(N, 0);
        for (int fc = 0; fc < 6; ++fc) {
            face_kind[fc] = c.periodic[fc / 2] ? FACE_PERIODIC : FACE_WALL;
            face_rho[fc][0] = face_rho[fc][1] = 1.0;
            face_u[fc][0] = face_u[fc][1] = face_u[fc][2] = 0.0;
        }
        for (int k = 0; k < c.n_components; ++k) {
            f[k].assign((size_t)q * N, T(0));
            fstar[k].assign((size_t)q * N, T(0));
            rho[k].assign(N, T(0));
            psi[k].assign(N, T(0));
            U[k].assign(N, T(0));
            for (int a = 0; a < 3; ++a) { j[k][a].assign(N, T(0)); F[k][a].assign(N, T(0)); }
        }
        for (int a = 0; a < 3; ++a) ucom[a].assign(N, T(0));
        rebuild_boundary_solids();
    }

    // ---- R9: MRT basis from polynomials of e_i (paper prints no M).
    // D2Q9 moment order (rho,e,eps,jx,qx,jy,qy,pxx,pxy) as in Eq. 15;
    // D3Q19: d'Humieres et al. (2002).  M^-1 = M^T diag(1/||row||^2) (rows orthogonal).
    void build_mrt() {
        double Md[19][19];
        for (int i = 0; i < q; ++i) {
            double cx = e[i][0], cy = e[i][1], cz = e[i][2];
            double c2 = cx * cx + cy * cy + cz * cz;
            if (d == 2) {
                Md[0][i] = 1;
                Md[1][i] = -4 + 3 * c2;
                Md[2][i] = 4 - 21 * c2 / 2 + 9 * c2 * c2 / 2;
                Md[3][i] = cx;
                Md[4][i] = (-5 + 3 * c2) * cx;
                Md[5][i] = cy;
                Md[6][i] = (-5 + 3 * c2) * cy;
                Md[7][i] = cx * cx - cy * cy;
                Md[8][i] = cx * cy;
            } else {
                Md[0][i] = 1;
                Md[1][i] = 19 * c2 - 30;
                Md[2][i] = (21 * c2 * c2 - 53 * c2 + 24) / 2;
                Md[3][i] = cx;
                Md[4][i] = (5 * c2 - 9) * cx;
                Md[5][i] = cy;
                Md[6][i] = (5 * c2 - 9) * cy;
                Md[7][i] = cz;
                Md[8][i] = (5 * c2 - 9) * cz;
                Md[9][i] = 3 * cx * cx - c2;
                Md[10][i] = (3 * c2 - 5) * (3 * cx * cx - c2);
                Md[11][i] = cy * cy - cz * cz;
                Md[12][i] = (3 * c2 - 5) * (cy * cy - cz * cz);
                Md[13][i] = cx * cy;
                Md[14][i] = cy * cz;
                Md[15][i] = cx * cz;
                Md[16][i] = (cy * cy - cz * cz) * cx;
                Md[17][i] = (cz * cz - cx * cx) * cy;
                Md[18][i] = (cx * cx - cy * cy) * cz;
            }
        }
        for (int r = 0; r < q; ++r) {
            double nrm = 0;
            for (int i = 0; i < q; ++i) nrm += Md[r][i] * Md[r][i];
            for (int i = 0; i < q; ++i) {
                M[r][i] = (T)Md[r][i];
                Minv[i][r] = (T)(Md[r][i] / nrm);
            }
        }
    }

    // ---- index helpers -------------------------------------------------
    int64_t idx(int x, int y, int z) const { return x + (int64_t)c.nx * (y + (int64_t)c.ny * z); }
    void coords(int64_t id, int* xyz) const {
        xyz[0] = (int)(id % c.nx);
        xyz[1] = (int)((id / c.nx) % c.ny);
        xyz[2] = (int)(id / ((int64_t)c.nx * c.ny));
    }
    // Neighbour used by the scalar stencils (S2, S4): periodic axes wrap, non-periodic
    // axes clamp the index (zero-gradient; R10).
    int64_t scalar_nbr(const int* xyz, int dir) const {
        int p[3];
        for (int a = 0; a < 3; ++a) {
            int v = xyz[a] + e[dir][a];
            if (v < 0) v = c.periodic[a] ? v + n[a] : 0;
            if (v >= n[a]) v = c.periodic[a] ? v - n[a] : n[a] - 1;
            p[a] = v;
        }
        return idx(p[0], p[1], p[2]);
    }
    // Source of the pull x - e_i (S7).  Returns -1-face if the link crosses a
    // non-periodic face (lowest axis wins), else the wrapped source index.
    int64_t pull_source(const int* xyz, int dir) const {
        int p[3];
        int crossed = -1;
        for (int a = 0; a < 3; ++a) {
            int v = xyz[a] - e[dir][a];
            if (v < 0) {
                if (c.periodic[a]) v += n[a];
                else { if (crossed < 0) crossed = 2 * a; v = 0; }
            } else if (v >= n[a]) {
                if (c.periodic[a]) v -= n[a];
                else { if (crossed < 0) crossed = 2 * a + 1; v = n[a] - 1; }
            }
            p[a] = v;
        }
        if (crossed >= 0) return -1 - crossed;
        return idx(p[0], p[1], p[2]);
    }

    void rebuild_boundary_solids() {
        bsolid.clear();
        for (int64_t id = 0; id < N; ++id) {
            if (!solid[id]) continue;
            int xyz[3];
            coords(id, xyz);
            bool any = false;
            for (int i = 1; i < q; ++i)
                if (!solid[scalar_nbr(xyz, i)]) { any = true; break; }
            if (any) bsolid.push_back(id);
        }
    }

    int set_solid_mask(const uint8_t* m) override {
        for (int64_t id = 0; id < N; ++id) solid[id] = m[id] ? 1 : 0;
        rebuild_boundary_solids();
        return 0;
    }

    int set_face_bc(int face, int kind, const double* rho_w, const double* u_w) override {
        if (face < 0 || face >= 2 * d) return -1;
        if (c.periodic[face / 2]) return -1;
        if (kind != FACE_WALL && kind != FACE_VELOCITY && kind != FACE_PRESSURE) return -1;
        face_kind[face] = kind;
        for (int k = 0; k < 2; ++k) face_rho[face][k] = rho_w ? rho_w[k] : 1.0;
        for (int a = 0; a < 3; ++a) face_u[face][a] = u_w ? u_w[a] : 0.0;
        return 0;
    }

    // Relaxation time of the momentum of component k: tau_k for BGK; for MRT 1 / (rate of the momentum rows), which
    // need not be 1/s_nu.  It is this time that enters the common velocity (R6) and the velocity shift (R7):
    // only then does a collision change the total momentum by exactly sum_k F^k (Eq. 3 + Eq. 10).
    T momentum_time(int k) const {
        if (c.collision == COLL_MRT) return T(1) / (T)c.mrt_rates[k][3];
        return (T)c.tau[k];
    }

    // ---- f_eq (R1): w_i rho [1 + e.u/cs2 + (e.u)^2/(2 cs2^2) - u.u/(2 cs2)]
    T feq(int i, T r, const T* u) const {
        T eu = T(0), uu = T(0);
        for (int a = 0; a < d; ++a) { eu += (T)e[i][a] * u[a]; uu += u[a] * u[a]; }
        return wT[i] * r * (T(1) + eu / cs2 + eu * eu / (T(2) * cs2 * cs2) - uu / (T(2) * cs2));
    }

    T load_f(int k, int i, int64_t id) const {
        T s = f[k][(size_t)i * N + id];
        if (c.rho_ref != 0.0) s += (T)(w[i] * c.rho_ref);
        return s;
    }
    T to_store(int i, T v) const {
        if (c.rho_ref != 0.0) v -= (T)(w[i] * c.rho_ref);
        return round_store<T>(v, c.store_dtype);
    }

    // ---- S0: f = f_eq(rho0, u0); solid cells hold f_eq(1,0) and are never updated
    // (P:195-199 initialisation; "zero velocity").
    int init_fields(const double* const* rho0, const double* u0) override {
        for (int k = 0; k < c.n_components; ++k) {
            for (int64_t id = 0; id < N; ++id) {
                T u[3] = {T(0), T(0), T(0)};
                T r = T(1);
                if (!solid[id]) {
                    r = (T)rho0[k][id];
                    if (u0) for (int a = 0; a < d; ++a) u[a] = (T)u0[(size_t)a * N + id];
                }
                for (int i = 0; i < q; ++i) f[k][(size_t)i * N + id] = to_store(i, feq(i, r, u));
            }
        }
        steps_done = 0;
        return 0;
    }

    // ---- S3: pseudopotential (Eq. 12; R4: radicand clamped at 0; P:275 psi=rho;
    // P:349 psi=exp(-1/rho); SC93 psi = rho0(1-exp(-rho/rho0)), reading R15).
    T pseudopotential(int k, T r) const {
        int kind = c.psi_kind[k];
        if (kind == PSI_RHO) return r;
        if (kind == PSI_EXP) return r > T(0) ? std::exp(-T(1) / r) : T(0);
        if (kind == PSI_SC93) { T r0 = (T)c.rho0[k]; return r0 * (T(1) - std::exp(-r / r0)); }
        T Tc = (T)eos_critical_temperature(kind, c.eos_a[k], c.eos_b[k], c.eos_R[k]);
        T p = eos_pressure<T>(kind, (T)c.eos_a[k], (T)c.eos_b[k], (T)c.eos_R[k], (T)c.eos_omega[k],
                              (T)c.eos_T[k], Tc, r);
        T rad = T(2) * ((T)c.alpha[k] * p - cs2 * r) / (T)c.G[k][k];
        return rad > T(0) ? std::sqrt(rad) : T(0);
    }

    // Eq. 12, second line: U^k = alpha^k p_EOS^k - c_s^2 rho^k (EOS kinds only; the Zhang-Chen term needs an EOS)
    T zc_potential(int k, T r) const {
        int kind = c.psi_kind[k];
        if (kind > PSI_EOS_RKS) return T(0);
        T Tc = (T)eos_critical_temperature(kind, c.eos_a[k], c.eos_b[k], c.eos_R[k]);
        T p = eos_pressure<T>(kind, (T)c.eos_a[k], (T)c.eos_b[k], (T)c.eos_R[k], (T)c.eos_omega[k],
                              (T)c.eos_T[k], Tc, r);
        return (T)c.alpha[k] * p - cs2 * r;
    }

    // S1..S4: moments, virtual density, psi, force -- everything S6 needs.
    void compute_fields() {
        const int nc = c.n_components;
        // S1 (Eq. 4 / Eq. 10): rho = sum_i f_i, j = sum_i f_i e_i
        for (int k = 0; k < nc; ++k) {
#pragma omp parallel for schedule(static) if (N >= 262144)
            for (int64_t id = 0; id < N; ++id) {
                if (solid[id]) {
                    rho[k][id] = T(0); psi[k][id] = T(0);
                    for (int a = 0; a < 3; ++a) { j[k][a][id] = T(0); F[k][a][id] = T(0); }
                    continue;
                }
                T r = T(0), jj[3] = {T(0), T(0), T(0)};
                for (int i = 0; i < q; ++i) {
                    T fi = load_f(k, i, id);
                    r += fi;
                    for (int a = 0; a < d; ++a) jj[a] += fi * (T)e[i][a];
                }
                rho[k][id] = r;
                for (int a = 0; a < 3; ++a) j[k][a][id] = jj[a];
            }
        }
        // S2 (Eq. 17 + limiter; R11, R12): virtual density at boundary solids
        for (int k = 0; k < nc; ++k) {
            for (size_t b = 0; b < bsolid.size(); ++b) {
                int64_t id = bsolid[b];
                int xyz[3];
                coords(id, xyz);
                T num = T(0), den = T(0);
                for (int i = 1; i < q; ++i) {
                    int64_t nb = scalar_nbr(xyz, i);
                    if (solid[nb]) continue;
                    num += wT[i] * rho[k][nb];
                    den += wT[i];
                }
                T rs = (T)c.wet_phi[k] * (num / den) - (T)c.wet_drho[k];
                if (rs < (T)c.wet_lo[k]) rs = (T)c.wet_lo[k];
                if (rs > (T)c.wet_hi[k]) rs = (T)c.wet_hi[k];
                rho[k][id] = rs;
            }
        }
        // S3: psi at fluid cells and boundary solids; all other solids keep psi = 0
        for (int k = 0; k < nc; ++k) {
#pragma omp parallel for schedule(static) if (N >= 262144)
            for (int64_t id = 0; id < N; ++id)
                if (!solid[id]) psi[k][id] = pseudopotential(k, rho[k][id]);
            for (size_t b = 0; b < bsolid.size(); ++b) psi[k][bsolid[b]] = pseudopotential(k, rho[k][bsolid[b]]);
            if (c.zc_A[k] != 0.0) {
                for (int64_t id = 0; id < N; ++id)
                    if (!solid[id]) U[k][id] = zc_potential(k, rho[k][id]);
                for (size_t b = 0; b < bsolid.size(); ++b) U[k][bsolid[b]] = zc_potential(k, rho[k][bsolid[b]]);
            }
        }
        // S4 (Eq. 13 F_SC; wetting folded in through psi(rho_s)):
        // F^k(x) = -psi^k(x) sum_k' g_kk' sum_i G_i psi^k'(x+e_i) e_i,  G_i = w_i/c_s^2 (R2)
        for (int k = 0; k < nc; ++k) {
#pragma omp parallel for schedule(static) if (N >= 262144)
            for (int64_t id = 0; id < N; ++id) {
                if (solid[id]) continue;
                int xyz[3];
                coords(id, xyz);
                T acc[3] = {T(0), T(0), T(0)};
                for (int kp = 0; kp < nc; ++kp) {
                    T s[3] = {T(0), T(0), T(0)};
                    for (int i = 1; i < q; ++i) {
                        T v = gw[i] * psi[kp][scalar_nbr(xyz, i)];
                        for (int a = 0; a < d; ++a) s[a] += v * (T)e[i][a];
                    }
                    for (int a = 0; a < d; ++a) acc[a] += (T)c.G[k][kp] * s[a];
                }
                for (int a = 0; a < 3; ++a) F[k][a][id] = -psi[k][id] * acc[a];
                // Eq. 13: F^k = A_kk F_ZC^k + (1 - A_kk) F_SC^k,  F_ZC^k = -sum_i G_i U^k(x+e_i) e_i
                if (c.zc_A[k] != 0.0) {
                    T z[3] = {T(0), T(0), T(0)};
                    for (int i = 1; i < q; ++i) {
                        T v = gw[i] * U[k][scalar_nbr(xyz, i)];
                        for (int a = 0; a < d; ++a) z[a] += v * (T)e[i][a];
                    }
                    const T A = (T)c.zc_A[k];
                    for (int a = 0; a < 3; ++a) F[k][a][id] = A * (-z[a]) + (T(1) - A) * F[k][a][id];
                }
                // body force driving the flow: the same acceleration on every component (R19)
                for (int a = 0; a < d; ++a)
                    if (c.body_accel[a] != 0.0) F[k][a][id] += rho[k][id] * (T)c.body_accel[a];
            }
        }
        // S5 (R6): common velocity u' = sum_k (j^k/tau_k) / sum_k (rho^k/tau_k); = j/rho for one component
        // (tau_k = momentum_time(k))
#pragma omp parallel for schedule(static) if (N >= 262144)
        for (int64_t id = 0; id < N; ++id) {
            if (solid[id]) { for (int a = 0; a < 3; ++a) ucom[a][id] = T(0); continue; }
            if (nc == 1) {
                for (int a = 0; a < 3; ++a) ucom[a][id] = j[0][a][id] / rho[0][id];
            } else {
                T den = T(0), num[3] = {T(0), T(0), T(0)};
                for (int k = 0; k < nc; ++k) {
                    den += rho[k][id] / momentum_time(k);
                    for (int a = 0; a < 3; ++a) num[a] += j[k][a][id] / momentum_time(k);
                }
                for (int a = 0; a < 3; ++a) ucom[a][id] = num[a] / den;
            }
        }
    }

    // S6: collision + forcing at every fluid cell -> fstar
    void collide() {
        const int nc = c.n_components;
        for (int k = 0; k < nc; ++k) {
            const T tau = (T)c.tau[k];
#pragma omp parallel for schedule(static) if (N >= 262144)
            for (int64_t id = 0; id < N; ++id) {
                if (solid[id]) continue;
                T fi[19], fe[19], fs[19];
                for (int i = 0; i < q; ++i) fi[i] = load_f(k, i, id);
                if (c.no_collide) {
                    for (int i = 0; i < q; ++i) fstar[k][(size_t)i * N + id] = fi[i];
                    continue;
                }
                T r = rho[k][id];
                T u[3] = {ucom[0][id], ucom[1][id], ucom[2][id]};
                T du[3];  // Eq. 5: Delta u = F dt / rho
                for (int a = 0; a < 3; ++a) du[a] = F[k][a][id] / r;
                T ueq[3] = {u[0], u[1], u[2]};
                if (c.forcing == FORCE_SHIFT)  // R7: u_eq = u' + tau F/rho, no source term
                    for (int a = 0; a < 3; ++a) ueq[a] = u[a] + momentum_time(k) * du[a];
                for (int i = 0; i < q; ++i) fe[i] = feq(i, r, ueq);
                if (c.collision == COLL_BGK) {
                    // Eq. 3 line 1
                    for (int i = 0; i < q; ++i) fs[i] = fi[i] - (fi[i] - fe[i]) / tau;
                } else {
                    // Eq. 3 line 2: f* = f - M^-1 S M (f - f_eq)
                    T neq[19], m[19];
                    for (int i = 0; i < q; ++i) neq[i] = fi[i] - fe[i];
                    for (int r_ = 0; r_ < q; ++r_) {
                        T s = T(0);
                        for (int i = 0; i < q; ++i) s += M[r_][i] * neq[i];
                        m[r_] = (T)c.mrt_rates[k][r_] * s;
                    }
                    for (int i = 0; i < q; ++i) {
                        T s = T(0);
                        for (int r_ = 0; r_ < q; ++r_) s += Minv[i][r_] * m[r_];
                        fs[i] = fi[i] - s;
                    }
                    // Eq. 14-16: surface-tension control, D2Q9.  Source C in moment space (Eq. 15, moment
                    // order rho,e,eps,jx,qx,jy,qy,pxx,pxy), Q from the pseudopotential (Eq. 16, reading R20)
                    if (c.st_kappa[k] != 0.0 && d == 2) {
                        int xyz[3];
                        coords(id, xyz);
                        const T A = (T)c.zc_A[k], ps0 = psi[k][id];
                        T Qxx = T(0), Qyy = T(0), Qxy = T(0);
                        for (int i = 1; i < q; ++i) {
                            const T ps1 = psi[k][scalar_nbr(xyz, i)];
                            const T v = gw[i] * ((T(1) - A) * ps0 * (ps1 - ps0) + T(0.5) * A * (ps1 * ps1 - ps0 * ps0));
                            Qxx += v * (T)(e[i][0] * e[i][0]);
                            Qyy += v * (T)(e[i][1] * e[i][1]);
                            Qxy += v * (T)(e[i][0] * e[i][1]);
                        }
                        // R20: Eq. 16 as printed has no interaction strength; with the factor g_kk (= -1) the
                        // tension falls as 1 - kappa, without it it would rise
                        const T qn = (T)c.st_kappa[k] * (T)c.G[k][k];
                        Qxx *= qn; Qyy *= qn; Qxy *= qn;
                        T C[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
                        C[1] = T(1.5) * (T)c.mrt_rates[k][1] * (Qxx + Qyy);
                        C[2] = -T(1.5) * (T)c.mrt_rates[k][2] * (Qxx + Qyy);
                        C[7] = -(T)c.mrt_rates[k][7] * (Qxx - Qyy);
                        C[8] = -(T)c.mrt_rates[k][8] * Qxy;
                        for (int i = 0; i < q; ++i) {
                            T s = T(0);
                            for (int r_ = 0; r_ < q; ++r_) s += Minv[i][r_] * C[r_];
                            fs[i] += s;
                        }
                    }
                }
                if (c.forcing == FORCE_EDM) {
                    // Eq. 5: f* += f_eq(rho, u+du) - f_eq(rho, u)   (R8: bare u')
                    T up[3] = {u[0] + du[0], u[1] + du[1], u[2] + du[2]};
                    for (int i = 0; i < q; ++i) fs[i] += feq(i, r, up) - fe[i];
                }
                for (int i = 0; i < q; ++i) fstar[k][(size_t)i * N + id] = fs[i];
            }
        }
    }

    // S7 (Eq. 2; halfway bounce-back R13; inlet/outlet R10): pull streaming
    void stream() {
        const int nc = c.n_components;
        for (int k = 0; k < nc; ++k) {
#pragma omp parallel for schedule(static) if (N >= 262144)
            for (int64_t id = 0; id < N; ++id) {
                if (solid[id]) continue;
                int xyz[3];
                coords(id, xyz);
                for (int i = 0; i < q; ++i) {
                    int64_t src = pull_source(xyz, i);
                    T v;
                    if (src < 0) {
                        int face = (int)(-1 - src);
                        T bounced = fstar[k][(size_t)opp[i] * N + id];
                        if (face_kind[face] == FACE_VELOCITY) {
                            // f_i = f*_ibar + 2 w_i rho_w (e_i.u_w)/cs2
                            T eu = T(0);
                            for (int a = 0; a < d; ++a) eu += (T)e[i][a] * (T)face_u[face][a];
                            v = bounced + T(2) * wT[i] * (T)face_rho[face][k] * eu / cs2;
                        } else if (face_kind[face] == FACE_PRESSURE) {
                            // f_i = -f*_ibar + 2 w_i rho_w [1 + (e_i.u)^2/(2 cs2^2) - u.u/(2 cs2)], u = node's own u'
                            T eu = T(0), uu = T(0);
                            for (int a = 0; a < d; ++a) {
                                eu += (T)e[i][a] * ucom[a][id];
                                uu += ucom[a][id] * ucom[a][id];
                            }
                            v = -bounced + T(2) * wT[i] * (T)face_rho[face][k]
                                               * (T(1) + eu * eu / (T(2) * cs2 * cs2) - uu / (T(2) * cs2));
                        } else {
                            v = bounced;  // wall face: halfway bounce-back
                        }
                    } else if (solid[src]) {
                        v = fstar[k][(size_t)opp[i] * N + id];  // halfway bounce-back (R13)
                    } else {
                        v = fstar[k][(size_t)i * N + src];
                    }
                    f[k][(size_t)i * N + id] = to_store(i, v);
                }
            }
        }
    }

    int step(int nsteps) override {
        for (int s = 0; s < nsteps; ++s) {
            compute_fields();
            collide();
            stream();
            ++steps_done;
        }
        return 0;
    }

    // S8 (Eq. 6): rho^k; u = (sum_k j^k + 1/2 sum_k F^k)/sum_k rho^k;
    // p = cs2 sum rho^k + 1/2 sum_kk' g_kk' psi^k psi^k'
    int get_macroscopic(double* const* rho_out, double* u_out, double* p_out) override {
        compute_fields();
        const int nc = c.n_components;
        for (int64_t id = 0; id < N; ++id) {
            for (int k = 0; k < nc; ++k)
                if (rho_out && rho_out[k]) rho_out[k][id] = (double)rho[k][id];
            if (solid[id]) {
                if (u_out) for (int a = 0; a < d; ++a) u_out[(size_t)a * N + id] = 0.0;
                if (p_out) p_out[id] = 0.0;
                continue;
            }
            T rt = T(0);
            for (int k = 0; k < nc; ++k) rt += rho[k][id];
            if (u_out) {
                for (int a = 0; a < d; ++a) {
                    T js = T(0), Fs = T(0);
                    for (int k = 0; k < nc; ++k) { js += j[k][a][id]; Fs += F[k][a][id]; }
                    u_out[(size_t)a * N + id] = (double)((js + Fs / T(2)) / rt);
                }
            }
            if (p_out) {
                T pp = T(0);
                for (int k = 0; k < nc; ++k)
                    for (int kp = 0; kp < nc; ++kp) pp += (T)c.G[k][kp] * psi[k][id] * psi[kp][id];
                p_out[id] = (double)(cs2 * rt + pp / T(2));
            }
        }
        return 0;
    }

    int get_populations(int k, double* out) override {
        if (k < 0 || k >= c.n_components) return -1;
        for (int i = 0; i < q; ++i)
            for (int64_t id = 0; id < N; ++id) out[(size_t)i * N + id] = (double)load_f(k, i, id);
        return 0;
    }
    int set_populations(int k, const double* in) override {
        if (k < 0 || k >= c.n_components) return -1;
        for (int i = 0; i < q; ++i)
            for (int64_t id = 0; id < N; ++id) f[k][(size_t)i * N + id] = to_store(i, (T)in[(size_t)i * N + id]);
        return 0;
    }

    // bit i (1 <= i < q) set  <=>  the pull of direction i at this fluid cell does NOT
    // read a fluid neighbour (source solid, or across a non-periodic face).
    // Solid cells report exactly 0x80000000.  Integer-only; compared bit-exactly
    // with the CUDA path.
    int get_link_flags(uint32_t* out) override {
        for (int64_t id = 0; id < N; ++id) {
            uint32_t fl = 0;
            if (solid[id]) { out[id] = 0x80000000u; continue; }
            int xyz[3];
            coords(id, xyz);
            for (int i = 1; i < q; ++i) {
                int64_t src = pull_source(xyz, i);
                if (src < 0 || solid[src]) fl |= (1u << i);
            }
            out[id] = fl;
        }
        return 0;
    }
    int64_t get_boundary_solids(int64_t* out, int64_t cap) override {
        int64_t m = (int64_t)bsolid.size();
        if (out) for (int64_t b = 0; b < m && b < cap; ++b) out[b] = bsolid[b];
        return m;
    }
    int get_force(int k, double* out) override {
        compute_fields();
        for (int a = 0; a < d; ++a)
            for (int64_t id = 0; id < N; ++id) out[(size_t)a * N + id] = (double)F[k][a][id];
        return 0;
    }
    int get_psi(int k, double* out) override {
        compute_fields();
        for (int64_t id = 0; id < N; ++id) out[id] = (double)psi[k][id];
        return 0;
    }
};

bool config_ok(const olbm_config& c) {
    if (c.lattice != LAT_D2Q9 && c.lattice != LAT_D3Q19) return false;
    if (c.nx < 1 || c.ny < 1 || c.nz < 1) return false;
    if (c.lattice == LAT_D2Q9 && c.nz != 1) return false;
    if (c.n_components < 1 || c.n_components > 2) return false;
    if (c.compute_dtype != DT_F32 && c.compute_dtype != DT_F64) return false;
    if (c.compute_dtype == DT_F32 && c.store_dtype == DT_F64) return false;
    if (c.compute_dtype == DT_F64 && c.store_dtype == DT_F16) return false;
    for (int k = 0; k < c.n_components; ++k) {
        if (c.psi_kind[k] < 0 || c.psi_kind[k] > PSI_SC93) return false;
        if (c.psi_kind[k] <= PSI_EOS_RKS && !(c.G[k][k] < 0.0)) return false;  // R4: g_kk < 0 under the root
        if (!(c.tau[k] > 0.5)) return false;
        if (c.collision == COLL_MRT) {   // the momentum rows share one non-zero rate (momentum_time)
            const int nj = c.lattice == LAT_D2Q9 ? 2 : 3;
            if (!(c.mrt_rates[k][3] > 0.0)) return false;
            for (int a = 1; a < nj; ++a)
                if (c.mrt_rates[k][3 + 2 * a] != c.mrt_rates[k][3]) return false;
        }
    }
    return true;
}

}  // namespace

extern "C" {

void* olbm_create(const olbm_config* cfg) {
    if (!cfg || !config_ok(*cfg)) return nullptr;
    if (cfg->compute_dtype == DT_F64) return new Sim<double>(*cfg);
    return new Sim<float>(*cfg);
}
void olbm_destroy(void* h) { delete static_cast<SimBase*>(h); }
int olbm_set_solid_mask(void* h, const uint8_t* m) { return static_cast<SimBase*>(h)->set_solid_mask(m); }
int olbm_set_face_bc(void* h, int face, int kind, const double* rho_w, const double* u_w) {
    return static_cast<SimBase*>(h)->set_face_bc(face, kind, rho_w, u_w);
}
int olbm_init_fields(void* h, const double* const* rho, const double* u) {
    return static_cast<SimBase*>(h)->init_fields(rho, u);
}
int olbm_step(void* h, int n) { return static_cast<SimBase*>(h)->step(n); }
int olbm_get_macroscopic(void* h, double* const* rho, double* u, double* p) {
    return static_cast<SimBase*>(h)->get_macroscopic(rho, u, p);
}
int olbm_get_populations(void* h, int k, double* out) { return static_cast<SimBase*>(h)->get_populations(k, out); }
int olbm_set_populations(void* h, int k, const double* in) { return static_cast<SimBase*>(h)->set_populations(k, in); }
int olbm_get_link_flags(void* h, uint32_t* out) { return static_cast<SimBase*>(h)->get_link_flags(out); }
int64_t olbm_get_boundary_solids(void* h, int64_t* out, int64_t cap) {
    return static_cast<SimBase*>(h)->get_boundary_solids(out, cap);
}
int olbm_get_force(void* h, int k, double* out) { return static_cast<SimBase*>(h)->get_force(k, out); }
int olbm_get_psi(void* h, int k, double* out) { return static_cast<SimBase*>(h)->get_psi(k, out); }

// Stand-alone pieces exposed so the pins can reach them directly.
int olbm_lattice(int lattice, int* q_out, int* e_out /*[q][3]*/, double* w_out /*[q]*/, int* opp_out /*[q]*/) {
    int q = lattice == LAT_D2Q9 ? 9 : 19;
    const int (*e)[3] = lattice == LAT_D2Q9 ? E_D2Q9 : E_D3Q19;
    const double* w = lattice == LAT_D2Q9 ? W_D2Q9 : W_D3Q19;
    *q_out = q;
    for (int i = 0; i < q; ++i) {
        for (int a = 0; a < 3; ++a) e_out[3 * i + a] = e[i][a];
        w_out[i] = w[i];
        for (int k = 0; k < q; ++k)
            if (e[k][0] == -e[i][0] && e[k][1] == -e[i][1] && e[k][2] == -e[i][2]) opp_out[i] = k;
    }
    return 0;
}
// f_eq of one cell, fp64 (lattice, rho, u[3]) -> out[q]
int olbm_feq(int lattice, double rho, const double* u, double* out) {
    olbm_config c;
    std::memset(&c, 0, sizeof c);
    c.lattice = lattice; c.nx = c.ny = c.nz = 1; c.n_components = 1;
    c.compute_dtype = DT_F64; c.store_dtype = DT_F64; c.tau[0] = 1.0; c.psi_kind[0] = PSI_RHO;
    Sim<double> s(c);
    for (int i = 0; i < s.q; ++i) out[i] = s.feq(i, rho, u);
    return s.q;
}
// MRT matrices (fp64): M[q][q], Minv[q][q] row-major
int olbm_mrt_matrices(int lattice, double* M, double* Minv) {
    olbm_config c;
    std::memset(&c, 0, sizeof c);
    c.lattice = lattice; c.nx = c.ny = c.nz = 1; c.n_components = 1;
    c.compute_dtype = DT_F64; c.store_dtype = DT_F64; c.tau[0] = 1.0; c.psi_kind[0] = PSI_RHO;
    Sim<double> s(c);
    for (int r = 0; r < s.q; ++r)
        for (int i = 0; i < s.q; ++i) { M[r * s.q + i] = s.M[r][i]; Minv[r * s.q + i] = s.Minv[r][i]; }
    return s.q;
}
double olbm_eos_critical_temperature(int kind, double a, double b, double R) {
    return eos_critical_temperature(kind, a, b, R);
}
// p_EOS(rho) for an array of densities (fp64)
int olbm_eos_pressure(int kind, double a, double b, double R, double omega, double T, const double* rho,
                      double* p, int64_t n) {
    double Tc = eos_critical_temperature(kind, a, b, R);
    for (int64_t i = 0; i < n; ++i) p[i] = eos_pressure<double>(kind, a, b, R, omega, T, Tc, rho[i]);
    return 0;
}
float olbm_round_to_half(float v) { return round_to_half(v); }
int olbm_set_threads(int nthreads) {
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    return omp_get_max_threads();
#else
    (void)nthreads;
    return 1;
#endif
}
int olbm_config_size() { return (int)sizeof(olbm_config); }

}  // extern "C"
