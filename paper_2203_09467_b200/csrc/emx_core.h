// emx_core.h -- constants, device-side parameter block and the counter-based RNG.
//
// Everything under csrc/ is written from the paper's description of the loop
// and the readings in DESIGN.md section 3; it shares no source with oracle/.
// Functions are marked EMX_HD so that a developer can also compile them for the host in a
// scratch harness; the library itself only ever instantiates them inside __global__ kernels.
#pragma once
#include <stdint.h>
#include <math.h>
#include "../../include/emx.h"

#if defined(__CUDACC__)
#define EMX_HD __host__ __device__ __forceinline__
// the larger building blocks (samplers, propagation, lookups).  Out-of-line copies were tried against the
// instruction-fetch stalls of the first fused kernel and lost to the call ABI and spills:
// everything is inlined, and one kernel per pool and phase keeps the code small instead
#define EMX_NI __host__ __device__ __forceinline__
#else
#define EMX_HD inline
#define EMX_NI inline
#endif

namespace emx {

// CODATA 2018 (C1)
constexpr double kMe = 0.51099895000;       // electron mass, MeV
constexpr double kRe = 2.8179403262e-13;    // classical electron radius, cm
constexpr double kAlpha = 7.2973525693e-3;  // fine-structure constant
constexpr double kNa = 6.02214076e23;       // Avogadro, 1/mol
constexpr double kCB = 2.99792458;          // curvature [1/cm] = q * kCB * B[T] / p[MeV/c] (r = 0.33356 cm at 1 MeV/c, 1 T)
constexpr double kPi = 3.14159265358979323846;
constexpr double kInf = __builtin_huge_val(); // +inf

enum : int { kGamma = 0, kElectron = 1, kPositron = 2 };

struct Material {
    int n_elem;
    int Z[EMX_MAX_ELEM];
    double A[EMX_MAX_ELEM], w[EMX_MAX_ELEM], n_i[EMX_MAX_ELEM];
    double rho, I, n_e, hwp, X0, Tcut, kcut;
};

struct Volume {
    int n_faces;
    int surf[EMX_MAX_FACES];
    int sense[EMX_MAX_FACES];
    int material, tally;
};

// One face of a cell with everything the navigation needs in one 16-byte word: the cells' face lists resolved
// against the surface table once, on the host (faces[vol * EMX_MAX_FACES + i]; n of face 0 = faces of the cell)
struct Face {
    double v;      // plane position or cylinder radius
    int S;         // surface id
    int8_t type;   // EMX_S_*
    int8_t sense;  // side of the surface the cell is on
    int16_t n;     // face 0 only: low byte = number of faces of the cell, high byte = how many of them are planes (they come first)
};

// Read-only problem data ("params" in the paper's params/state split), passed to
// kernels by value; the pointers refer to the problem's one small device block.
struct Params {
    emx_physics ph;
    int n_mat, n_surf, n_vol, n_tally;
    const Material *mat;
    const int *surf_type;
    const double *surf_v;
    const Volume *vol;
    const Face *faces;      // [n_vol][EMX_MAX_FACES]
    const double *tab;      // [n_mat][EMX_NTABLE][n_E]
    const int *nb_off;      // neighbour candidates: cells having face (S, sense); index 2*S + (sense > 0)
    const int *nb_list;
    const int *nb2_off;     // per (S, sense): cells that do not list S at all (the only other cells that can match)
    const int *nb2_list;
    double Bmag, Bhat[3];
    double field_eps_floor;       // ph.field_eps / 3125: the error below which a substep grows by the full factor 5 (C9)
    int field_kind;               // 0 uniform; 1 solenoid with fringe (emx_set_field_fringe)
    double fringe_z0, fringe_a;   // cm
    double lnE0, dlnE, inv_dlnE;  // grid: x_j = lnE0 + j * dlnE
};

// libm calls of the step path, out of line (one copy each instead of one per call site)
EMX_NI double m_log(double x) { return log(x); }
EMX_NI double m_exp(double x) { return exp(x); }
EMX_NI double m_pow(double x, double y) { return pow(x, y); }
EMX_NI double m_cbrt(double x) { return cbrt(x); }
EMX_NI void m_sincos(double a, double &s, double &c) {
#if defined(__CUDA_ARCH__)
    sincos(a, &s, &c);
#else
    s = sin(a);
    c = cos(a);
#endif
}

struct Vec3 {
    double x, y, z;
};
EMX_HD Vec3 operator+(Vec3 a, Vec3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
EMX_HD Vec3 operator-(Vec3 a, Vec3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
EMX_HD Vec3 operator*(double s, Vec3 a) { return {s * a.x, s * a.y, s * a.z}; }
EMX_HD double norm(Vec3 a) { return sqrt(a.x * a.x + a.y * a.y + a.z * a.z); }
EMX_HD double comp(const Vec3 &a, int i) { return i == 0 ? a.x : (i == 1 ? a.y : a.z); }

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) -- DESIGN.md C2.  PAPER.md:189 used XORWOW;
// BASELINE.json north_star asks for a counter-based Philox keyed by track id and step.
struct Philox4 {
    uint32_t w[4];
};

EMX_NI Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return {{c0, c1, c2, c3}};
}

// 52-bit uniform strictly inside (0,1): (k + 1/2) 2^-52, k in [0, 2^52)
EMX_HD double u01(uint32_t hi, uint32_t lo) {
    const uint64_t k = (((uint64_t)hi << 32) | (uint64_t)lo) >> 12;
    return ((double)k + 0.5) * (1.0 / 4503599627370496.0);
}

// Draw cursor of one (seed, primary, track id, step): key = (seed32, prim),
// counter = (draw block, step, tid_lo, tid_hi); draw n uses block n/2, words 2(n%2), 2(n%2)+1.
struct Rng {
    uint32_t k0, k1, step, tlo, thi;
    uint32_t n;          // next draw number
    uint32_t w2, w3;     // second half of the current block (valid when n is odd)

    EMX_HD void init(uint64_t seed, uint32_t prim, uint64_t tid, uint32_t step_) {
        k0 = (uint32_t)seed;
        k1 = prim;
        step = step_;
        tlo = (uint32_t)tid;
        thi = (uint32_t)(tid >> 32);
        n = 0;
        w2 = w3 = 0;
    }
    EMX_HD double next() {
        double v;
        if ((n & 1u) == 0u) {
            const Philox4 b = philox4x32_10(n >> 1, step, tlo, thi, k0, k1);
            w2 = b.w[2];
            w3 = b.w[3];
            v = u01(b.w[0], b.w[1]);
        } else {
            v = u01(w2, w3);
        }
        ++n;
        return v;
    }
};

// stand-alone draw (level-1 hook) and child track ids
EMX_HD double draw_at(uint64_t seed, uint32_t prim, uint64_t tid, uint32_t step, uint32_t n) {
    const Philox4 b = philox4x32_10(n >> 1, step, (uint32_t)tid, (uint32_t)(tid >> 32), (uint32_t)seed, prim);
    return (n & 1u) ? u01(b.w[2], b.w[3]) : u01(b.w[0], b.w[1]);
}
EMX_HD uint64_t child_tid(uint32_t k0, uint32_t prim, uint64_t tid, uint32_t step, uint32_t ordinal) {
    const Philox4 b = philox4x32_10(0xFFFFFFFFu - ordinal, step, (uint32_t)tid, (uint32_t)(tid >> 32), k0, prim);
    return ((uint64_t)b.w[0] << 32) | (uint64_t)b.w[1];
}

}  // namespace emx
