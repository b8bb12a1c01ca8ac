// mi_oracle.cpp -- plain, slow, obviously-correct CPU oracle for the exhaustive MI map.
//
// *** TEST INFRASTRUCTURE, NOT PRODUCT CODE. ***
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code, header, table or constant with the CUDA
// library under paper_1909_10690_b200/csrc; neither side includes or imports the other.
//
// What it computes (Vianna & Murta 2019, PAPER.md):
//   * the "Transform" block v(T(x)) of Fig. 1            (section 1)
//   * the joint histogram over ALL fixed voxels          (section 4: "uses all the
//     voxels and produces a full histogram")
//   * Shannon entropies and MI, eq. 1 and eq. 2
//   * Tsallis MI from the SAME histogram                 (section 4)
//   * the exhaustive map over a 3-parameter family, one value per parameter triple, and its
//     arg max, eq. 3
//
// The method is exact (a histogram and sums over it), so the oracle is the plain definition.
// Because the north-star demands BIT-EXACT nearest-neighbour histograms, the definition includes
// the floating-point operation sequence wherever a rounding decides a voxel or a bin; those
// sequences are the "CANON-n" readings of SURVEY.md section 8(c), restated in DESIGN.md.  The
// paper does not fix a precision (reading A16): coordinates and samples are fp32,
// counts are integers, entropies are fp64.  orc_joint_hist_f64 does the geometry in fp64 so the
// effect of that reading can be reported (pin P12).
//
// Partial-volume interpolation (reading A21; Maes et al., the paper's ref. [5], PAPER.md:228;
// "the effects of interpolation") is orc_joint_hist_pv below, pinned by
// tests/test_oracle_pv_pins.py (PV1..PV7).
//
// Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): P1..P12 of DESIGN.md.  The one point with
// no pin is the sign/character of Tsallis maps versus the paper's figures -- "parity unpinned"
// (the paper prints no Tsallis formula; reading A1/A2).
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off [-mfma] -fopenmp -shared -fPIC (oracle/build.py).
// -ffp-contract=off matters: every fmaf below is an explicit fused op, every other a*b+c is two
// roundings.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Geometry {
    int32_t fd[3];   // fixed dims (nx, ny, nz), x fastest in memory
    int32_t md[3];   // moving dims
};

// CANON-5 binning: uniform bins over [lo, hi], hi lands in the last bin, clamp outside.
inline float bin_scale(int nb, float lo, float hi) {
    return (float)((double)nb / ((double)hi - (double)lo));
}
inline int bin_of(float v, float lo, float scale, int nb) {
    float d = v - lo;            // one rounding
    float t = d * scale;         // one rounding
    float f = floorf(t);
    f = fmaxf(f, 0.0f);
    f = fminf(f, (float)(nb - 1));
    return (int)f;
}

// CANON-2 coordinates: continuous moving index of fixed voxel (ix, iy, iz).
inline void coords(const float M[12], int ix, int iy, int iz, float c[3]) {
    for (int k = 0; k < 3; ++k) {
        float r = fmaf(M[k * 4 + 1], (float)iy, fmaf(M[k * 4 + 2], (float)iz, M[k * 4 + 3]));
        c[k] = fmaf(M[k * 4 + 0], (float)ix, r);
    }
}

// CANON-3 nearest neighbour.  Returns false if the sample is outside the moving volume.
inline bool sample_nn(const float* mv, const int32_t md[3], const float c[3], float* out) {
    int j[3];
    for (int k = 0; k < 3; ++k) {
        float r = floorf(c[k] + 0.5f);                       // round half up
        if (!(r >= 0.0f && r < (float)md[k])) return false;  // tested in float
        j[k] = (int)r;
    }
    *out = mv[((size_t)j[2] * md[1] + j[1]) * md[0] + j[0]];
    return true;
}

inline float lerp(float p, float q, float f) {
    float d = q - p;             // rounded to fp32 first
    return fmaf(f, d, p);
}

// CANON-4 trilinear: x-lerps, then y-lerps, then the z-lerp.
inline bool sample_tri(const float* mv, const int32_t md[3], const float c[3], float* out) {
    int i0[3], i1[3];
    float f[3];
    for (int k = 0; k < 3; ++k) {
        if (!(c[k] >= -0.5f && c[k] < (float)md[k] - 0.5f)) return false;
        float g = floorf(c[k]);
        f[k] = c[k] - g;
        int gi = (int)g;
        i0[k] = gi > 0 ? gi : 0;
        i1[k] = (gi + 1 < md[k] - 1) ? gi + 1 : md[k] - 1;
    }
    const size_t nx = md[0], ny = md[1];
    auto at = [&](int x, int y, int z) { return mv[((size_t)z * ny + y) * nx + x]; };
    float v00 = lerp(at(i0[0], i0[1], i0[2]), at(i1[0], i0[1], i0[2]), f[0]);
    float v10 = lerp(at(i0[0], i1[1], i0[2]), at(i1[0], i1[1], i0[2]), f[0]);
    float v01 = lerp(at(i0[0], i0[1], i1[2]), at(i1[0], i0[1], i1[2]), f[0]);
    float v11 = lerp(at(i0[0], i1[1], i1[2]), at(i1[0], i1[1], i1[2]), f[0]);
    float w0 = lerp(v00, v10, f[1]);
    float w1 = lerp(v01, v11, f[1]);
    *out = lerp(w0, w1, f[2]);
    return true;
}

// CANON-7, eq. 1: H = -sum_{p>0} p ln p over a vector of counts with total N.
double shannon_of_counts(const double* cnt, size_t n, double N) {
    double H = 0.0;
    for (size_t i = 0; i < n; ++i) {
        if (cnt[i] > 0.0) {
            double p = cnt[i] / N;
            H -= p * std::log(p);
        }
    }
    return H;
}
// Tsallis entropy S_q = (1 - sum_{p>0} p^q) / (q - 1)   (reading A1).
double tsallis_of_counts(const double* cnt, size_t n, double N, double q) {
    double s = 0.0;
    for (size_t i = 0; i < n; ++i) {
        if (cnt[i] > 0.0) s += std::pow(cnt[i] / N, q);
    }
    return (1.0 - s) / (q - 1.0);
}

}  // namespace

extern "C" {

// CANON-1: physical transform y = A x + t (x fixed-physical mm, y moving-physical mm,
// direction per eq. 3) composed with the two volume-centred geometries into the
// index-space map c = M i + m0, evaluated in double left to right, then rounded to fp32.
// T is row-major 3x4 [A|t]; out is row-major 3x4 [M|m0].
void orc_index_affine(const double T[12], const int32_t fd[3], const double fs[3],
                      const int32_t md[3], const double ms[3], float out[12]) {
    double hf[3], hm[3];
    for (int k = 0; k < 3; ++k) {
        hf[k] = ((double)fd[k] - 1.0) / 2.0;
        hm[k] = ((double)md[k] - 1.0) / 2.0;
    }
    for (int r = 0; r < 3; ++r) {
        double M[3];
        for (int c = 0; c < 3; ++c) {
            double a = T[r * 4 + c] * fs[c];
            M[c] = a / ms[r];
        }
        double m0 = T[r * 4 + 3] / ms[r];
        m0 = m0 - M[0] * hf[0];
        m0 = m0 - M[1] * hf[1];
        m0 = m0 - M[2] * hf[2];
        m0 = m0 + hm[r];
        for (int c = 0; c < 3; ++c) out[r * 4 + c] = (float)M[c];
        out[r * 4 + 3] = (float)m0;
    }
}

// Family generators: parameter triple -> physical 3x4 [A|t].
//   0 translation (mm), 1 Euler degrees R = Rz(p2) Ry(p1) Rx(p0), 2 versor (ball of radius 1,
//   PAPER.md:121), 3 scale factors, 4 log-scale (zero-centred).
int orc_family_matrix(int family, const double p[3], double T[12]) {
    for (int i = 0; i < 12; ++i) T[i] = 0.0;
    T[0] = T[5] = T[10] = 1.0;
    switch (family) {
    case 0:
        T[3] = p[0]; T[7] = p[1]; T[11] = p[2];
        return 0;
    case 1: {
        const double d2r = 3.14159265358979323846 / 180.0;
        double cx = std::cos(p[0] * d2r), sx = std::sin(p[0] * d2r);
        double cy = std::cos(p[1] * d2r), sy = std::sin(p[1] * d2r);
        double cz = std::cos(p[2] * d2r), sz = std::sin(p[2] * d2r);
        double Rx[9] = {1, 0, 0, 0, cx, -sx, 0, sx, cx};
        double Ry[9] = {cy, 0, sy, 0, 1, 0, -sy, 0, cy};
        double Rz[9] = {cz, -sz, 0, sz, cz, 0, 0, 0, 1};
        double RyRx[9], R[9];
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) {
                double s = 0.0;
                for (int k = 0; k < 3; ++k) s += Ry[i * 3 + k] * Rx[k * 3 + j];
                RyRx[i * 3 + j] = s;
            }
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) {
                double s = 0.0;
                for (int k = 0; k < 3; ++k) s += Rz[i * 3 + k] * RyRx[k * 3 + j];
                R[i * 3 + j] = s;
            }
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) T[i * 4 + j] = R[i * 3 + j];
        return 0;
    }
    case 2: {
        double x = p[0], y = p[1], z = p[2];
        double n2 = x * x + y * y + z * z;
        if (n2 > 1.0) {  // outside the unit ball -> mapped to its surface
            double n = std::sqrt(n2);
            x /= n; y /= n; z /= n;
            n2 = x * x + y * y + z * z;
        }
        double w2 = 1.0 - n2;
        double w = w2 > 0.0 ? std::sqrt(w2) : 0.0;
        // rotation matrix of the unit quaternion (w, x, y, z)
        T[0] = 1.0 - 2.0 * (y * y + z * z); T[1] = 2.0 * (x * y - w * z); T[2] = 2.0 * (x * z + w * y);
        T[4] = 2.0 * (x * y + w * z); T[5] = 1.0 - 2.0 * (x * x + z * z); T[6] = 2.0 * (y * z - w * x);
        T[8] = 2.0 * (x * z - w * y); T[9] = 2.0 * (y * z + w * x); T[10] = 1.0 - 2.0 * (x * x + y * y);
        return 0;
    }
    case 3:
        T[0] = p[0]; T[5] = p[1]; T[10] = p[2];
        return 0;
    case 4:
        T[0] = std::exp(p[0]); T[5] = std::exp(p[1]); T[10] = std::exp(p[2]);
        return 0;
    default:
        return 1;
    }
}

// CANON-5 applied to a whole volume (step a1 "prebin").  out[i] in [0, nb-1].
void orc_prebin(const float* vol, int64_t n, int nb, float lo, float hi, int32_t* out) {
    const float scale = bin_scale(nb, lo, hi);
    for (int64_t i = 0; i < n; ++i) out[i] = bin_of(vol[i], lo, scale, nb);
}

// The Transform block alone: value[i] = v(T(x_i)) for every fixed voxel, valid[i] = 1 if the
// sample is inside the moving volume.  interp: 0 nearest, 1 trilinear.
void orc_resample(const int32_t fd[3], const float* moving, const int32_t md[3], const float M[12],
                  int interp, float* value, uint8_t* valid) {
    for (int iz = 0; iz < fd[2]; ++iz)
        for (int iy = 0; iy < fd[1]; ++iy)
            for (int ix = 0; ix < fd[0]; ++ix) {
                size_t i = ((size_t)iz * fd[1] + iy) * fd[0] + ix;
                float c[3], v = 0.0f;
                coords(M, ix, iy, iz, c);
                bool ok = interp ? sample_tri(moving, md, c, &v) : sample_nn(moving, md, c, &v);
                value[i] = ok ? v : 0.0f;
                valid[i] = ok ? 1 : 0;
            }
}

// CANON-6: joint histogram h[a*nb + b] of (bin u(x), bin v(T(x))) over every fixed voxel whose
// sample is inside the moving volume (reading A5).  Returns the number of valid samples.
// mask (may be NULL): one byte per fixed voxel; voxels with mask == 0 take no part (reading A19: the
// random-sampling question of PAPER.md:212 -- the sampled subset is an INPUT, drawn by the harness).
int64_t orc_joint_hist_masked(const float* fixed, const int32_t fd[3], const float* moving,
                              const int32_t md[3], const float M[12], int nb, float flo, float fhi,
                              float mlo, float mhi, int interp, const uint8_t* mask, uint32_t* hist) {
    std::memset(hist, 0, sizeof(uint32_t) * (size_t)nb * nb);
    const float fscale = bin_scale(nb, flo, fhi);
    const float mscale = bin_scale(nb, mlo, mhi);
    int64_t nvalid = 0;
    for (int iz = 0; iz < fd[2]; ++iz)
        for (int iy = 0; iy < fd[1]; ++iy)
            for (int ix = 0; ix < fd[0]; ++ix) {
                float c[3], v;
                size_t i = ((size_t)iz * fd[1] + iy) * fd[0] + ix;
                if (mask != nullptr && mask[i] == 0) continue;
                coords(M, ix, iy, iz, c);
                bool ok = interp ? sample_tri(moving, md, c, &v) : sample_nn(moving, md, c, &v);
                if (!ok) continue;
                int a = bin_of(fixed[i], flo, fscale, nb);
                int b = bin_of(v, mlo, mscale, nb);
                hist[(size_t)a * nb + b] += 1;
                ++nvalid;
            }
    return nvalid;
}

int64_t orc_joint_hist(const float* fixed, const int32_t fd[3], const float* moving,
                       const int32_t md[3], const float M[12], int nb, float flo, float fhi,
                       float mlo, float mhi, int interp, uint32_t* hist) {
    return orc_joint_hist_masked(fixed, fd, moving, md, M, nb, flo, fhi, mlo, mhi, interp, nullptr, hist);
}

// Pin P12: the same histogram with ALL geometry in fp64 (index-space matrix M64 given in double,
// coordinates, weights and interpolation in double; binning of the fp64 sample in double).
// Reported, never gated.
int64_t orc_joint_hist_f64(const float* fixed, const int32_t fd[3], const float* moving,
                           const int32_t md[3], const double M[12], int nb, float flo, float fhi,
                           float mlo, float mhi, int interp, uint32_t* hist) {
    std::memset(hist, 0, sizeof(uint32_t) * (size_t)nb * nb);
    const float fscale = bin_scale(nb, flo, fhi);
    const double mscale = (double)nb / ((double)mhi - (double)mlo);
    int64_t nvalid = 0;
    const size_t nx = md[0], ny = md[1];
    auto at = [&](int x, int y, int z) { return (double)moving[((size_t)z * ny + y) * nx + x]; };
    for (int iz = 0; iz < fd[2]; ++iz)
        for (int iy = 0; iy < fd[1]; ++iy)
            for (int ix = 0; ix < fd[0]; ++ix) {
                double c[3];
                bool ok = true;
                for (int k = 0; k < 3; ++k) {
                    c[k] = M[k * 4 + 0] * ix + M[k * 4 + 1] * iy + M[k * 4 + 2] * iz + M[k * 4 + 3];
                    if (!(c[k] >= -0.5 && c[k] < (double)md[k] - 0.5)) ok = false;
                }
                if (!ok) continue;
                double v;
                if (interp == 0) {
                    int j[3];
                    for (int k = 0; k < 3; ++k) {
                        j[k] = (int)std::floor(c[k] + 0.5);
                        if (j[k] > md[k] - 1) j[k] = md[k] - 1;
                    }
                    v = at(j[0], j[1], j[2]);
                } else {
                    int i0[3], i1[3];
                    double f[3];
                    for (int k = 0; k < 3; ++k) {
                        double g = std::floor(c[k]);
                        f[k] = c[k] - g;
                        int gi = (int)g;
                        i0[k] = gi > 0 ? gi : 0;
                        i1[k] = (gi + 1 < md[k] - 1) ? gi + 1 : md[k] - 1;
                    }
                    auto L = [](double p, double q, double t) { return p + t * (q - p); };
                    double v00 = L(at(i0[0], i0[1], i0[2]), at(i1[0], i0[1], i0[2]), f[0]);
                    double v10 = L(at(i0[0], i1[1], i0[2]), at(i1[0], i1[1], i0[2]), f[0]);
                    double v01 = L(at(i0[0], i0[1], i1[2]), at(i1[0], i0[1], i1[2]), f[0]);
                    double v11 = L(at(i0[0], i1[1], i1[2]), at(i1[0], i1[1], i1[2]), f[0]);
                    v = L(L(v00, v10, f[1]), L(v01, v11, f[1]), f[2]);
                }
                size_t i = ((size_t)iz * fd[1] + iy) * fd[0] + ix;
                int a = bin_of(fixed[i], flo, fscale, nb);
                double t = std::floor((v - (double)mlo) * mscale);
                if (t < 0.0) t = 0.0;
                if (t > (double)(nb - 1)) t = (double)(nb - 1);
                hist[(size_t)a * nb + (int)t] += 1;
                ++nvalid;
            }
    return nvalid;
}

}  // extern "C"

namespace {

// CANON-7 on a table of counts (uint32 voxel counts, or uint64 partial-volume weight units -- the
// probabilities h/N do not depend on the unit).
template <typename CountT>
void entropies_of(const CountT* hist, int nb, const double* q, int nq, int form, double* out, double* detail) {
    std::vector<double> joint((size_t)nb * nb), pa(nb, 0.0), pb(nb, 0.0);
    double N = 0.0;
    for (int a = 0; a < nb; ++a)
        for (int b = 0; b < nb; ++b) {
            double c = (double)hist[(size_t)a * nb + b];
            joint[(size_t)a * nb + b] = c;
            pa[a] += c;
            pb[b] += c;
            N += c;
        }
    if (N <= 0.0) {
        for (int i = 0; i < 1 + nq; ++i) out[i] = 0.0;
        if (detail) detail[0] = detail[1] = detail[2] = 0.0;
        return;
    }
    double HA = shannon_of_counts(pa.data(), nb, N);
    double HB = shannon_of_counts(pb.data(), nb, N);
    double HAB = shannon_of_counts(joint.data(), joint.size(), N);
    double I = HA + HB - HAB;  // eq. 2
    out[0] = I;
    if (detail) { detail[0] = HA; detail[1] = HB; detail[2] = HAB; }
    for (int k = 0; k < nq; ++k) {
        if (q[k] == 1.0) { out[1 + k] = I; continue; }
        double SA = tsallis_of_counts(pa.data(), nb, N, q[k]);
        double SB = tsallis_of_counts(pb.data(), nb, N, q[k]);
        double SAB = tsallis_of_counts(joint.data(), joint.size(), N, q[k]);
        double Iq = SA + SB - SAB;
        if (form == 1) Iq += (1.0 - q[k]) * SA * SB;
        out[1 + k] = Iq;
    }
}

}  // namespace

extern "C" {

// CANON-7: joint histogram -> [Shannon I, I_q0, I_q1, ...]  (eq. 1-2; Tsallis per
// reading A1).  form 0 = ADDITIVE, 1 = PSEUDO_ADDITIVE.  detail (may be NULL) receives
// [H(A), H(B), H(A,B)].  Empty histogram -> all zeros (reading A13).
void orc_entropies(const uint32_t* hist, int nb, const double* q, int nq, int form, double* out,
                   double* detail) {
    entropies_of(hist, nb, q, nq, form, out, detail);
}
void orc_entropies_u64(const uint64_t* hist, int nb, const double* q, int nq, int form, double* out,
                       double* detail) {
    entropies_of(hist, nb, q, nq, form, out, detail);
}

// Partial-volume interpolation (reading A21).  The method of Maes et al. (ref. [5] of the paper,
// PAPER.md:228) interpolates no intensity: the sample point's eight neighbours n_i of the moving grid
// each add their trilinear weight w_i (sum 1) to the cell (bin u(x), bin v(n_i)).  The paper only
// names the problem ("we start to see the effects of interpolation") and the open
// question about bins; the arithmetic is this build's reading:
//   * coordinates, validity region, floor / fraction and the edge clamp are CANON-2 and CANON-4;
//   * the fraction f_k of each axis is rounded to 1/32 voxel, u_k = floor(32 f_k + 0.5) in 0..32
//     (both fp32 operations are exact or a single rounding), and the weight of the neighbour with
//     offsets (dx,dy,dz) is the integer (dx ? u_x : 32-u_x)(dy ? u_y : 32-u_y)(dz ? u_z : 32-u_z):
//     the eight weights of a sample sum to 2^15 exactly, every histogram is an exact integer table
//     independent of summation order, and 2^15 units are one voxel;
//   * neighbours of weight 0 are skipped; the neighbour's bin is CANON-5 of its own value.
// Returns the number of valid samples; sum(hist) = 2^15 * that number.
int64_t orc_joint_hist_pv(const float* fixed, const int32_t fd[3], const float* moving, const int32_t md[3],
                          const float M[12], int nb, float flo, float fhi, float mlo, float mhi,
                          const uint8_t* mask, uint64_t* hist) {
    std::memset(hist, 0, sizeof(uint64_t) * (size_t)nb * nb);
    const float fscale = bin_scale(nb, flo, fhi);
    const float mscale = bin_scale(nb, mlo, mhi);
    const size_t nx = md[0], ny = md[1];
    int64_t nvalid = 0;
    for (int iz = 0; iz < fd[2]; ++iz)
        for (int iy = 0; iy < fd[1]; ++iy)
            for (int ix = 0; ix < fd[0]; ++ix) {
                size_t i = ((size_t)iz * fd[1] + iy) * fd[0] + ix;
                if (mask != nullptr && mask[i] == 0) continue;
                float c[3];
                coords(M, ix, iy, iz, c);
                int idx[3][2];   // the two neighbours per axis, clamped to the volume
                int w[3][2];     // their weights in 1/32
                bool ok = true;
                for (int k = 0; k < 3; ++k) {
                    if (!(c[k] >= -0.5f && c[k] < (float)md[k] - 0.5f)) { ok = false; break; }
                    float g = floorf(c[k]);
                    float f = c[k] - g;
                    int u = (int)floorf(f * 32.0f + 0.5f);
                    int gi = (int)g;
                    idx[k][0] = gi > 0 ? gi : 0;
                    idx[k][1] = (gi + 1 < md[k] - 1) ? gi + 1 : md[k] - 1;
                    w[k][0] = 32 - u;
                    w[k][1] = u;
                }
                if (!ok) continue;
                int a = bin_of(fixed[i], flo, fscale, nb);
                for (int dz = 0; dz < 2; ++dz)
                    for (int dy = 0; dy < 2; ++dy)
                        for (int dx = 0; dx < 2; ++dx) {
                            int wt = w[0][dx] * w[1][dy] * w[2][dz];
                            if (wt == 0) continue;
                            float v = moving[((size_t)idx[2][dz] * ny + idx[1][dy]) * nx + idx[0][dx]];
                            int b = bin_of(v, mlo, mscale, nb);
                            hist[(size_t)a * nb + b] += (uint64_t)wt;
                        }
                ++nvalid;
            }
    return nvalid;
}

// N transforms with partial-volume interpolation -> N x (1+nq) MI values (+ optional uint64
// histograms and valid counts); OpenMP over transforms as orc_eval_batch_masked.
int orc_eval_batch_pv(const float* fixed, const int32_t fd[3], const float* moving, const int32_t md[3],
                      const float* M, int64_t N, int nb, float flo, float fhi, float mlo, float mhi,
                      const double* q, int nq, int form, const uint8_t* mask, double* mi_out,
                      uint64_t* hist_out, int64_t* nvalid_out) {
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
#pragma omp parallel
    {
        std::vector<uint64_t> h((size_t)nb * nb);
#pragma omp for schedule(dynamic, 1)
        for (int64_t t = 0; t < N; ++t) {
            int64_t nv = orc_joint_hist_pv(fixed, fd, moving, md, M + t * 12, nb, flo, fhi, mlo, mhi, mask, h.data());
            orc_entropies_u64(h.data(), nb, q, nq, form, mi_out + t * (1 + nq), nullptr);
            if (hist_out) std::memcpy(hist_out + (size_t)t * nb * nb, h.data(), sizeof(uint64_t) * h.size());
            if (nvalid_out) nvalid_out[t] = nv;
        }
    }
    return nthreads;
}

// N index-space transforms -> N x (1+nq) MI values (+ optional histograms and valid counts).
// OpenMP over transforms, one private histogram per thread; this is the timed CPU baseline.
// Returns the number of threads used.
int orc_eval_batch_masked(const float* fixed, const int32_t fd[3], const float* moving, const int32_t md[3],
                          const float* M, int64_t N, int nb, float flo, float fhi, float mlo, float mhi,
                          int interp, const double* q, int nq, int form, const uint8_t* mask, double* mi_out,
                          uint32_t* hist_out, int64_t* nvalid_out) {
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
#pragma omp parallel
    {
        std::vector<uint32_t> h((size_t)nb * nb);
#pragma omp for schedule(dynamic, 1)
        for (int64_t t = 0; t < N; ++t) {
            int64_t nv = orc_joint_hist_masked(fixed, fd, moving, md, M + t * 12, nb, flo, fhi, mlo, mhi,
                                               interp, mask, h.data());
            orc_entropies(h.data(), nb, q, nq, form, mi_out + t * (1 + nq), nullptr);
            if (hist_out) std::memcpy(hist_out + (size_t)t * nb * nb, h.data(), sizeof(uint32_t) * h.size());
            if (nvalid_out) nvalid_out[t] = nv;
        }
    }
    return nthreads;
}

int orc_eval_batch(const float* fixed, const int32_t fd[3], const float* moving, const int32_t md[3],
                   const float* M, int64_t N, int nb, float flo, float fhi, float mlo, float mhi,
                   int interp, const double* q, int nq, int form, double* mi_out,
                   uint32_t* hist_out, int64_t* nvalid_out) {
    return orc_eval_batch_masked(fixed, fd, moving, md, M, N, nb, flo, fhi, mlo, mhi, interp, q, nq, form, nullptr,
                                 mi_out, hist_out, nvalid_out);
}

// Exhaustive map: grid value k on axis d is lo[d] + k (hi[d]-lo[d])/(n[d]-1);
// interp: 0 nearest, 1 trilinear, 2 partial volume.
// map_out is (1+nq) x n[2] x n[1] x n[0], channel-major, p0 fastest; argmax per channel with ties
// to the lowest linear index (eq. 3).  Returns the number of threads used.
int orc_map_masked(const float* fixed, const int32_t fd[3], const double fs[3], const float* moving,
                   const int32_t md[3], const double ms[3], int nb, float flo, float fhi, float mlo,
                   float mhi, int family, const double lo[3], const double hi[3], const int32_t n[3],
                   const double* q, int nq, int form, int interp, const uint8_t* mask, double* map_out,
                   int64_t* argmax_out) {
    const int64_t NT = (int64_t)n[0] * n[1] * n[2];
    std::vector<float> M((size_t)NT * 12);
    for (int k2 = 0; k2 < n[2]; ++k2)
        for (int k1 = 0; k1 < n[1]; ++k1)
            for (int k0 = 0; k0 < n[0]; ++k0) {
                int kk[3] = {k0, k1, k2};
                double p[3], T[12];
                for (int d = 0; d < 3; ++d)
                    p[d] = n[d] == 1 ? lo[d] : lo[d] + (double)kk[d] * (hi[d] - lo[d]) / (double)(n[d] - 1);
                orc_family_matrix(family, p, T);
                int64_t t = ((int64_t)k2 * n[1] + k1) * n[0] + k0;
                orc_index_affine(T, fd, fs, md, ms, M.data() + t * 12);
            }
    std::vector<double> mi((size_t)NT * (1 + nq));
    int nthreads = interp == 2
        ? orc_eval_batch_pv(fixed, fd, moving, md, M.data(), NT, nb, flo, fhi, mlo, mhi, q, nq, form, mask,
                            mi.data(), nullptr, nullptr)
        : orc_eval_batch_masked(fixed, fd, moving, md, M.data(), NT, nb, flo, fhi, mlo, mhi, interp,
                                q, nq, form, mask, mi.data(), nullptr, nullptr);
    for (int ch = 0; ch < 1 + nq; ++ch) {
        int64_t best = 0;
        for (int64_t t = 0; t < NT; ++t) {
            double v = mi[(size_t)t * (1 + nq) + ch];
            map_out[(size_t)ch * NT + t] = v;
            if (v > map_out[(size_t)ch * NT + best]) best = t;
        }
        if (argmax_out) argmax_out[ch] = best;
    }
    return nthreads;
}

int orc_map(const float* fixed, const int32_t fd[3], const double fs[3], const float* moving,
            const int32_t md[3], const double ms[3], int nb, float flo, float fhi, float mlo,
            float mhi, int family, const double lo[3], const double hi[3], const int32_t n[3],
            const double* q, int nq, int form, int interp, double* map_out, int64_t* argmax_out) {
    return orc_map_masked(fixed, fd, fs, moving, md, ms, nb, flo, fhi, mlo, mhi, family, lo, hi, n, q, nq, form,
                          interp, nullptr, map_out, argmax_out);
}

int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
