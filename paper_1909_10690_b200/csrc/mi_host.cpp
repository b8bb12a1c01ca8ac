// mi_host.cpp -- step a2 of the hot path on the host, in double: family parameters -> physical
// 3x4 [A|t] -> index-space fp32 3x4 [M|m0] (DESIGN.md CANON-1).  Compiled with -ffp-contract=off:
// the rounding sequence of m0 below is part of the contract that makes nearest-neighbour
// histograms bit-exact, so no a*b+c here may be fused.
#include <cmath>

#include "mi_internal.h"

namespace mi {

// Uniform-bin scale of DESIGN.md CANON-5: nb / (hi - lo) formed in double, rounded once.
float bin_scale(int nbins, float lo, float hi) {
    double w = static_cast<double>(hi) - static_cast<double>(lo);
    return static_cast<float>(static_cast<double>(nbins) / w);
}

static void set_identity(double T[12]) {
    for (int i = 0; i < 12; ++i) T[i] = 0.0;
    T[0] = T[5] = T[10] = 1.0;
}

static void matmul3(const double a[3][3], const double b[3][3], double c[3][3]) {
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double acc = 0.0;
            for (int k = 0; k < 3; ++k) acc += a[i][k] * b[k][j];
            c[i][j] = acc;
        }
}

// Nine-parameter transform of the multi-metric gradient (A18): y = R(a) S(s) x + t with
// p = (tx,ty,tz mm, ax,ay,az deg, sx,sy,sz), R = Rz Ry Rx as in MI_FAMILY_ROTATION_EULER_DEG.
int family_matrix(int family, const double p[3], double T[12]);
void compose_matrix(const double p[9], double T[12]) {
    family_matrix(MI_FAMILY_ROTATION_EULER_DEG, p + 3, T);
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) T[i * 4 + j] = T[i * 4 + j] * p[6 + j];   // column j scaled by s_j
        T[i * 4 + 3] = p[i];
    }
}

// Transform families of the maps (translation 3.1, rotation 3.2, scale 3.3).
int family_matrix(int family, const double p[3], double T[12]) {
    set_identity(T);
    switch (family) {
    case MI_FAMILY_TRANSLATION:
        T[3] = p[0];
        T[7] = p[1];
        T[11] = p[2];
        return 0;
    case MI_FAMILY_ROTATION_EULER_DEG: {
        const double rad = 3.14159265358979323846 / 180.0;
        const double ca = std::cos(p[0] * rad), sa = std::sin(p[0] * rad);
        const double cb = std::cos(p[1] * rad), sb = std::sin(p[1] * rad);
        const double cg = std::cos(p[2] * rad), sg = std::sin(p[2] * rad);
        const double rx[3][3] = {{1, 0, 0}, {0, ca, -sa}, {0, sa, ca}};
        const double ry[3][3] = {{cb, 0, sb}, {0, 1, 0}, {-sb, 0, cb}};
        const double rz[3][3] = {{cg, -sg, 0}, {sg, cg, 0}, {0, 0, 1}};
        double yx[3][3], r[3][3];
        matmul3(ry, rx, yx);
        matmul3(rz, yx, r);
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) T[i * 4 + j] = r[i][j];
        return 0;
    }
    case MI_FAMILY_ROTATION_VERSOR: {
        // The paper's rotation space is a ball of radius 1 whose outside is mapped to the surface
        // (PAPER.md:121): p is the vector part of a unit quaternion.
        double vx = p[0], vy = p[1], vz = p[2];
        double nn = vx * vx + vy * vy + vz * vz;
        if (nn > 1.0) {
            const double len = std::sqrt(nn);
            vx /= len;
            vy /= len;
            vz /= len;
            nn = vx * vx + vy * vy + vz * vz;
        }
        const double ww = 1.0 - nn;
        const double w = ww > 0.0 ? std::sqrt(ww) : 0.0;
        T[0] = 1.0 - 2.0 * (vy * vy + vz * vz);
        T[1] = 2.0 * (vx * vy - w * vz);
        T[2] = 2.0 * (vx * vz + w * vy);
        T[4] = 2.0 * (vx * vy + w * vz);
        T[5] = 1.0 - 2.0 * (vx * vx + vz * vz);
        T[6] = 2.0 * (vy * vz - w * vx);
        T[8] = 2.0 * (vx * vz - w * vy);
        T[9] = 2.0 * (vy * vz + w * vx);
        T[10] = 1.0 - 2.0 * (vx * vx + vy * vy);
        return 0;
    }
    case MI_FAMILY_SCALE:
        T[0] = p[0];
        T[5] = p[1];
        T[10] = p[2];
        return 0;
    case MI_FAMILY_SCALE_LOG:
        T[0] = std::exp(p[0]);
        T[5] = std::exp(p[1]);
        T[10] = std::exp(p[2]);
        return 0;
    default:
        return 1;
    }
}

// Hand-off from an exhaustive map to the registration loop (A22): the nine parameters
// (t [mm], Euler angles [deg], scale factors) of map node (k0,k1,k2) of a family's grid, identity elsewhere.
// Translation, Euler and scale nodes are copied; log-scale nodes become factors exp(p); a versor node becomes
// the Euler angles of its rotation matrix R = Rz Ry Rx: ay = -asin(R20), ax = atan2(R21, R22), az = atan2(R10, R00).
int seed_from_node(int family, const double p[3], double out[9]) {
    for (int i = 0; i < 9; ++i) out[i] = i < 6 ? 0.0 : 1.0;
    switch (family) {
    case MI_FAMILY_TRANSLATION: out[0] = p[0]; out[1] = p[1]; out[2] = p[2]; return 0;
    case MI_FAMILY_ROTATION_EULER_DEG: out[3] = p[0]; out[4] = p[1]; out[5] = p[2]; return 0;
    case MI_FAMILY_SCALE: out[6] = p[0]; out[7] = p[1]; out[8] = p[2]; return 0;
    case MI_FAMILY_SCALE_LOG: out[6] = std::exp(p[0]); out[7] = std::exp(p[1]); out[8] = std::exp(p[2]); return 0;
    case MI_FAMILY_ROTATION_VERSOR: {
        double T[12];
        family_matrix(family, p, T);
        const double deg = 180.0 / 3.14159265358979323846;
        double s = -T[8];
        if (s > 1.0) s = 1.0;
        if (s < -1.0) s = -1.0;
        out[4] = std::asin(s) * deg;
        out[3] = std::atan2(T[9], T[10]) * deg;
        out[5] = std::atan2(T[4], T[0]) * deg;
        return 0;
    }
    default: return 1;
    }
}

// CANON-1.  Voxel i of a volume (dims n, spacing s) sits at s*(i - h), h = (n-1)/2; a transform
// is y = A x + t from fixed-physical to moving-physical (direction of eq. 3).  The
// continuous moving index is c = M i + m0 with
//   M[r][c] = (A[r][c]*sf[c]) / sm[r]
//   m0[r]   = ((((t[r]/sm[r]) - M[r][0]*hf[0]) - M[r][1]*hf[1]) - M[r][2]*hf[2]) + hm[r]
// left to right in double, each of the 12 numbers then rounded to fp32.
void index_affine(const double T[12], const int32_t fd[3], const double fs[3], const int32_t md[3],
                  const double ms[3], float out[12]) {
    double half_f[3], half_m[3];
    for (int d = 0; d < 3; ++d) {
        half_f[d] = (static_cast<double>(fd[d]) - 1.0) / 2.0;
        half_m[d] = (static_cast<double>(md[d]) - 1.0) / 2.0;
    }
    for (int r = 0; r < 3; ++r) {
        double row[3];
        for (int c = 0; c < 3; ++c) {
            const double num = T[r * 4 + c] * fs[c];
            row[c] = num / ms[r];
        }
        double off = T[r * 4 + 3] / ms[r];
        for (int c = 0; c < 3; ++c) {
            const double prod = row[c] * half_f[c];
            off = off - prod;
        }
        off = off + half_m[r];
        out[r * 4 + 0] = static_cast<float>(row[0]);
        out[r * 4 + 1] = static_cast<float>(row[1]);
        out[r * 4 + 2] = static_cast<float>(row[2]);
        out[r * 4 + 3] = static_cast<float>(off);
    }
}

}  // namespace mi
