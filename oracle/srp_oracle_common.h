/*
 * srp_oracle_common.h -- TEST INFRASTRUCTURE ONLY (see oracle/README.md).
 *
 * Shared by the two translation units of the CPU oracle (mesh generators and
 * photon tracer).  Nothing under paper_2602_10712_b200/ includes this file and
 * this file includes nothing from there: the oracle and the CUDA path share no
 * code.  Plain C99, fp64, single-threaded.
 *
 * Contents: Philox4x32-10 (counter-based RNG), the 23-bit
 * uniform mapping (reading R4), small fp64 vector helpers and the branch-free
 * orthonormal basis (O-step 1; Duff et al. 2017 "Building an orthonormal
 * basis, revisited").
 */
#ifndef SRP_ORACLE_COMMON_H
#define SRP_ORACLE_COMMON_H

#include <math.h>
#include <stdint.h>

/* ---- Philox4x32-10 (Salmon et al. 2011), written out from its definition:
 * 10 rounds of  (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
 * key bumped by the Weyl constants between rounds.  Pinned by the known-answer
 * vectors in tests/golden/philox_kat.txt. */
static inline void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2],
                                     uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Reading R4: xi = ((x >> 9) + 0.5) * 2^-23 = (2m+1) * 2^-24 with m < 2^23:
 * strictly inside (0,1) and an odd 24-bit integer times 2^-24, hence exactly
 * representable in fp32 and fp64 alike (a 24-bit m would need 25 bits). */
static inline double orc_uniform(uint32_t x)
{
    return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0);
}

typedef struct { double x, y, z; } orc_v3;

static inline orc_v3 orc_mk(double x, double y, double z) { orc_v3 r = {x, y, z}; return r; }
static inline orc_v3 orc_add(orc_v3 a, orc_v3 b) { return orc_mk(a.x + b.x, a.y + b.y, a.z + b.z); }
static inline orc_v3 orc_sub(orc_v3 a, orc_v3 b) { return orc_mk(a.x - b.x, a.y - b.y, a.z - b.z); }
static inline orc_v3 orc_scale(orc_v3 a, double s) { return orc_mk(a.x * s, a.y * s, a.z * s); }
static inline double orc_dot(orc_v3 a, orc_v3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
static inline orc_v3 orc_cross(orc_v3 a, orc_v3 b)
{
    return orc_mk(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
static inline orc_v3 orc_normalize(orc_v3 a)
{
    double n = sqrt(orc_dot(a, a));
    return orc_mk(a.x / n, a.y / n, a.z / n);
}

/* O-step 1: orthonormal (u, v) perpendicular to the unit vector s.
 *   sign = copysign(1, s.z); a = -1/(sign + s.z); b = s.x*s.y*a
 *   u = (1 + sign*s.x^2*a, sign*b, -sign*s.x);  v = (b, sign + s.y^2*a, -s.y) */
static inline void orc_basis(orc_v3 s, orc_v3 *u, orc_v3 *v)
{
    double sign = copysign(1.0, s.z);
    double a = -1.0 / (sign + s.z);
    double b = s.x * s.y * a;
    *u = orc_mk(1.0 + sign * s.x * s.x * a, sign * b, -sign * s.x);
    *v = orc_mk(b, sign + s.y * s.y * a, -s.y);
}

#endif /* SRP_ORACLE_COMMON_H */
