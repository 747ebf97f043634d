/*
 * srp_oracle_trace.c -- TEST INFRASTRUCTURE ONLY.  CPU oracle, part 2 of 2:
 * the forward photon tracer for the solar-radiation-pressure force
 *     F(omega, theta) = int_M f(x, omega, theta) dx            (Eq. 3)
 * with the light-to-force map l2f = L <n,w_in>+ (-w_in - w_out f_r) / c
 * (Eq. 2), estimated by Monte-Carlo path tracing with BRDF
 * importance sampling, next-event estimation and multiple bounces
 * (PAPER.md:146-159), every ray tested against ALL triangles.
 *
 * Forward form (R1-R16): a parallel photon bundle of
 * pressure P = L/c leaves an emitter rectangle perpendicular to the sun
 * direction; momentum is deposited at every hit.  The steps below are numbered
 * as in DESIGN.md "O-steps".  fp64, single thread, no acceleration structure,
 * no blocking or reordering.  Only the facet-material lobe thresholds are
 * taken in fp32 (they decide an integer: which lobe) -- DESIGN.md R17.
 *
 * Torque (Eq. 4): tau = int_M (x - x_COM) x f(x) dx -- every
 * momentum deposit, made at hit point x, also contributes (x - x_COM) x deposit.
 *
 * Glossy specular lobe ("per-face Phong material parameters"; DESIGN.md
 * reading R23): a facet with shininess n >= 0 scatters its specular part into the Phong lobe cos^n about the
 * mirror direction, importance-sampled, directions below the facet's horizon rejected and redrawn.
 *
 * Pins (tests/test_oracle_*.py): Philox KAT, flat plate, convex polyhedron,
 * cannonball limit, occlusion, V-groove, perpendicular-plate form factor,
 * conservation, symmetries, N^-1/2 decay, estimator agreement; torque: off-centre
 * plate, two-plate windmill, centre-of-mass shift identity, centred sphere; glossy lobe (test_oracle_glossy.py):
 * mean cosine (n+1)/(n+2), mirror limit, lobe axis at oblique incidence, horizon rejection, bookkeeping.
 *
 * Direct / indirect split (Fig. 5 rows 3-4; "OursGridNB" = no bounces): F_direct = the
 * momentum deposited where sun light first meets the surface (depth 0), F_indirect = F - F_direct = everything
 * deposited by light that has been reflected at least once.  Pins (tests/test_oracle_split.py): convex body =>
 * indirect = 0; direct = the B = 0 force, photon by photon; direct = the shadow-ray surface quadrature of P12;
 * V-groove: direct and indirect each P A_p.
 */
#include <stdlib.h>
#include <string.h>
#include "srp_oracle_common.h"

typedef struct {
    unsigned long long launched, primary_miss, absorbed, escaped, capped, segments;
    unsigned long long hits_at_depth[16];
} orc_stats;

typedef struct {
    double solar_pressure;   /* P, N/m^2 */
    int sampler;             /* 0 stratified-jittered Morton grid, 1 i.i.d. */
    int deposit;             /* 0 expected-value, 1 analog */
    int no_caustics;         /* 1: a photon whose FIRST reflection is specular is not followed (its first-hit deposit
                                stays).  That is the light a backward path tracer with a delta sun cannot find
                                (srp_oracle_backward below); used only to cross-check the two estimators. */
} orc_options;

/* O-step 4: closest hit over ALL triangles with index != src.
 * Moller-Trumbore on (v0, e1, e2); accept det != 0, u >= 0, v >= 0, u+v <= 1,
 * t > 0; smallest t wins, ties -> smallest index (strict <). */
static long closest_hit(const double *v0, const double *e1, const double *e2, long T,
                        orc_v3 o, orc_v3 d, long src, double *t_out)
{
    long best = -1; double tbest = INFINITY;
    for (long f = 0; f < T; ++f) {
        if (f == src) continue;
        orc_v3 E1 = orc_mk(e1[3 * f], e1[3 * f + 1], e1[3 * f + 2]);
        orc_v3 E2 = orc_mk(e2[3 * f], e2[3 * f + 1], e2[3 * f + 2]);
        orc_v3 pv = orc_cross(d, E2);
        double det = orc_dot(E1, pv);
        if (det == 0.0) continue;
        double inv = 1.0 / det;
        orc_v3 tv = orc_sub(o, orc_mk(v0[3 * f], v0[3 * f + 1], v0[3 * f + 2]));
        double u = orc_dot(tv, pv) * inv;
        if (!(u >= 0.0)) continue;
        orc_v3 qv = orc_cross(tv, E1);
        double v = orc_dot(d, qv) * inv;
        if (!(v >= 0.0) || !(u + v <= 1.0)) continue;
        double t = orc_dot(E2, qv) * inv;
        if (!(t > 0.0)) continue;
        if (t < tbest) { tbest = t; best = f; }
    }
    *t_out = tbest;
    return best;
}

/* A momentum deposit dd made at point x: force total dp += dd, torque total dq += (x - xc) x dd (Eq. 4). */
static void orc_deposit(const double dd[3], orc_v3 x, orc_v3 xc, double dp[3], double dq[3])
{
    const orc_v3 r = orc_sub(x, xc);
    dp[0] += dd[0]; dp[1] += dd[1]; dp[2] += dd[2];
    dq[0] += r.y * dd[2] - r.z * dd[1];
    dq[1] += r.z * dd[0] - r.x * dd[2];
    dq[2] += r.x * dd[1] - r.y * dd[0];
}

typedef struct { const double *v0, *e1, *e2, *nrm; long T; const float *shin; } orc_geom;

/* O-steps 4-7 for ONE photon that starts at o along d (src = the triangle it leaves, -1 for none) with momentum
 * weight wph: closest hit, deposit (force total dp, torque total dq about xc), lobe selection, continuation,
 * until it is absorbed, escapes or has been reflected B times.  The lobe draw of the hit at `depth` uses the
 * Philox counter (i, j, k, (depth + 1) | cflag). */
static void trace_photon(const orc_geom *G, const float *mats, orc_v3 o, orc_v3 d, long src, double wph,
                         uint32_t i, uint32_t j, uint32_t k, uint32_t cflag, const uint32_t key[2],
                         const orc_options *opt, int B, orc_v3 xc, orc_stats *st, double dp[3], double dq[3],
                         int *first_hit, unsigned long long *sig, double *dp0 /* deposits at depth 0, or NULL */)
{
    int depth = 0;
    for (;;) {
        /* O-step 4 */
        double t;
        st->segments++;
        long f = closest_hit(G->v0, G->e1, G->e2, G->T, o, d, src, &t);
        if (depth == 0 && first_hit) *first_hit = (int)f;
        if (f < 0) {
            if (depth == 0) st->primary_miss++; else st->escaped++;
            break;
        }
        st->hits_at_depth[depth]++;
        *sig = *sig * 1000003ULL + (unsigned long long)(f + 1);
        /* O-step 5: facing normal, mirror direction, deposit. */
        orc_v3 n = orc_mk(G->nrm[3 * f], G->nrm[3 * f + 1], G->nrm[3 * f + 2]);
        orc_v3 nf = (orc_dot(n, d) > 0.0) ? orc_scale(n, -1.0) : n;
        double cost = -orc_dot(d, nf);
        orc_v3 refl = orc_add(d, orc_scale(nf, 2.0 * cost));
        orc_v3 x = orc_add(o, orc_scale(d, t));
        const double al = mats[3 * f], rs = mats[3 * f + 1], rd = mats[3 * f + 2];
        /* dd = this hit's momentum deposit, made at x; Eq. 4: torque += (x - x_COM) x dd */
        double dd[3] = { 0, 0, 0 };
        /* R23: shininess < 0 (or none given) = the ideal mirror of R5; >= 0 = Phong lobe cos^n about refl */
        const int glossy = G->shin != NULL && G->shin[f] >= 0.0f;
        if (opt->deposit == 0 && !glossy) {
            double a = al + rs + rd;
            dd[0] = wph * (a * d.x - rs * refl.x - (2.0 / 3.0) * rd * nf.x);
            dd[1] = wph * (a * d.y - rs * refl.y - (2.0 / 3.0) * rd * nf.y);
            dd[2] = wph * (a * d.z - rs * refl.z - (2.0 / 3.0) * rd * nf.z);
        }
        if (opt->deposit == 0 && glossy) {
            /* absorbed and diffuse parts in expectation at every hit; the specular part has no closed-form mean
             * once the horizon truncates the lobe: it is deposited as d - d' when that lobe is drawn (below) */
            double a = al + rd;
            dd[0] = wph * (a * d.x - (2.0 / 3.0) * rd * nf.x);
            dd[1] = wph * (a * d.y - (2.0 / 3.0) * rd * nf.y);
            dd[2] = wph * (a * d.z - (2.0 / 3.0) * rd * nf.z);
        }
        /* O-step 6: lobe selection (thresholds in fp32, R17). */
        uint32_t c2[4] = { i, j, k, (uint32_t)(depth + 1) | cflag }, y[4];
        orc_philox4x32_10(c2, key, y);
        const double z0 = orc_uniform(y[0]), z1 = orc_uniform(y[1]), z2 = orc_uniform(y[2]);
        const float th1 = mats[3 * f];
        const float th2 = mats[3 * f] + mats[3 * f + 1];
        orc_v3 dnew;
        if (z0 < (double)th1) {
            if (opt->deposit == 1) { dd[0] = wph * d.x; dd[1] = wph * d.y; dd[2] = wph * d.z; }
            orc_deposit(dd, x, xc, dp, dq);
            if (depth == 0 && dp0) { dp0[0] += dd[0]; dp0[1] += dd[1]; dp0[2] += dd[2]; }
            st->absorbed++;
            break;
        } else if (z0 < (double)th2 && !glossy) {
            dnew = refl;
            if (opt->no_caustics && depth == 0) {
                if (opt->deposit == 1) { dd[0] = wph * (d.x - dnew.x); dd[1] = wph * (d.y - dnew.y); dd[2] = wph * (d.z - dnew.z); }
                orc_deposit(dd, x, xc, dp, dq);
                if (dp0) { dp0[0] += dd[0]; dp0[1] += dd[1]; dp0[2] += dd[2]; }
                st->capped++;
                break;
            }
        } else if (z0 < (double)th2) {
            /* Phong lobe: cos(theta) = xi^(1/(n+1)) about refl, phi uniform; attempt a = 0 uses (z1, z2) of the
             * lobe draw, attempt a >= 1 words 1 and 2 of Philox(i, j, k, (depth + 1) | cflag | a << 8).  The local
             * sample is laid out in the facet's frame (t_u, t_v, nf) of R18 and carried to refl by the rotation
             * that takes nf to refl about nf x refl (1 + nf . refl >= 1: no singular direction).  A direction
             * with d' . nf <= 0 is rejected; after 8 rejections the photon takes refl itself. */
            const double ns = (double)G->shin[f];
            orc_v3 tu = orc_normalize(orc_mk(G->e1[3 * f], G->e1[3 * f + 1], G->e1[3 * f + 2]));
            orc_v3 tv = orc_cross(nf, tu);
            orc_v3 kx = orc_cross(nf, refl);
            const double cc = orc_dot(nf, refl);
            double u1 = z1, u2 = z2;
            dnew = refl;
            for (int a = 0; a < 8; ++a) {
                if (a > 0) {
                    uint32_t c3[4] = { i, j, k, (uint32_t)(depth + 1) | cflag | ((uint32_t)a << 8) }, w[4];
                    orc_philox4x32_10(c3, key, w);
                    u1 = orc_uniform(w[1]); u2 = orc_uniform(w[2]);
                }
                const double ct = pow(u2, 1.0 / (ns + 1.0)), sn = sqrt(fmax(0.0, 1.0 - ct * ct));
                const double phi = 6.283185307179586476925286766559 * u1;
                orc_v3 L = orc_add(orc_add(orc_scale(tu, sn * cos(phi)), orc_scale(tv, sn * sin(phi))), orc_scale(nf, ct));
                orc_v3 kL = orc_cross(kx, L);
                orc_v3 cand = orc_add(orc_add(L, kL), orc_scale(orc_cross(kx, kL), 1.0 / (1.0 + cc)));
                if (orc_dot(cand, nf) > 0.0) { dnew = cand; break; }
            }
            if (opt->deposit == 0) {
                dd[0] += wph * (d.x - dnew.x); dd[1] += wph * (d.y - dnew.y); dd[2] += wph * (d.z - dnew.z);
            }
        } else {
            double phi = 6.283185307179586476925286766559 * z1, rho = sqrt(z2);
            double lx = rho * cos(phi), ly = rho * sin(phi), lz = sqrt(1.0 - z2);
            /* tangent frame (R18): first edge of the facet and nf x edge -- defined by the
             * mesh itself, so it has no discontinuity that rounding noise in nf could trip
             * (the step-1 rule flips across nf.z = 0, where axis-aligned facets sit) */
            orc_v3 tu = orc_normalize(orc_mk(G->e1[3 * f], G->e1[3 * f + 1], G->e1[3 * f + 2]));
            orc_v3 tv = orc_cross(nf, tu);
            dnew = orc_add(orc_add(orc_scale(tu, lx), orc_scale(tv, ly)), orc_scale(nf, lz));
        }
        if (opt->deposit == 1) {
            dd[0] = wph * (d.x - dnew.x); dd[1] = wph * (d.y - dnew.y); dd[2] = wph * (d.z - dnew.z);
        }
        orc_deposit(dd, x, xc, dp, dq);
        if (depth == 0 && dp0) { dp0[0] += dd[0]; dp0[1] += dd[1]; dp0[2] += dd[2]; }
        /* O-step 7: depth cap. */
        if (depth == B) { st->capped++; break; }
        o = x; d = dnew; src = f; depth += 1;
    }
}

static void deinterleave(uint64_t i, uint32_t *cx, uint32_t *cy)
{
    uint32_t x = 0, y = 0;
    for (int b = 0; b < 32; ++b) {
        x |= (uint32_t)((i >> (2 * b)) & 1u) << b;
        y |= (uint32_t)((i >> (2 * b + 1)) & 1u) << b;
    }
    *cx = x; *cy = y;
}

/*
 * Forces of ONE design (index k in its batch -- k enters the Philox counter)
 * for S sun directions.
 *   verts float[T][3][3], mats float[T][3] = (alpha, rho_s, rho_d)
 *   sun_dirs float[S][3]: body -> sun (the paper's omega); any length > 0
 *   j0: global direction index of sun_dirs[0] (enters the Philox counter), so a
 *       caller can split the directions of a pair list over processes
 *   F double[S][3] newtons; sumsq double[S][3] = sum over photons of the squared
 *       per-photon momentum total (for the MC standard error), may be NULL
 *   stats accumulated over all S (zeroed here), may be NULL
 *   first_hit int32[S][N] primary-hit triangle (-1 miss), may be NULL
 *   path_sig uint64[S][N] bookkeeping for the divergent-ray count, may be NULL: sig = 0, then
 *       sig = sig*1000003 + (triangle index + 1) at every hit (mod 2^64)
 *   x_com double[3] centre of mass (Eq. 4), Tq double[S][3] torque in N m, tq_sumsq double[S][3]
 *       sum of squared per-photon torque totals: all three may be NULL (no torque)
 *   shininess float[T] or NULL: Phong exponent of each facet's specular lobe, < 0 = ideal mirror (R23)
 * Returns 0, or -1 on invalid arguments.
 */
static int forces_core(const float *verts, const float *mats, const float *shininess, long T, int k,
                       const float *sun_dirs, int S, int j0, long long N, int B,
                       unsigned long long seed, const orc_options *opt,
                       double *F, double *sumsq, orc_stats *stats, int *first_hit,
                       unsigned long long *path_sig, const double *x_com, double *Tq,
                       double *tq_sumsq, double *F_direct /* double[S][3] or NULL */)
{
    if (!verts || !mats || !sun_dirs || !F || !opt || T <= 0 || S <= 0 || N <= 0 || B < 0 || B > 15)
        return -1;
    int m = 0;
    if (opt->sampler == 0) {
        while ((1LL << m) < N) ++m;
        if ((1LL << m) != N) return -1;          /* stratified grid needs N = 2^m */
    }
    const double nx = (double)(1LL << ((m + 1) / 2)), ny = (double)(1LL << (m / 2));
    const double P = opt->solar_pressure;
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };

    double *v0 = malloc(sizeof(double) * 3 * T), *e1 = malloc(sizeof(double) * 3 * T),
           *e2 = malloc(sizeof(double) * 3 * T), *nrm = malloc(sizeof(double) * 3 * T);
    double lo[3] = { INFINITY, INFINITY, INFINITY }, hi[3] = { -INFINITY, -INFINITY, -INFINITY };
    for (long f = 0; f < T; ++f) {
        for (int c = 0; c < 3; ++c) {
            double a = verts[9 * f + c], b = verts[9 * f + 3 + c], cc = verts[9 * f + 6 + c];
            v0[3 * f + c] = a; e1[3 * f + c] = b - a; e2[3 * f + c] = cc - a;
            double mn = fmin(a, fmin(b, cc)), mx = fmax(a, fmax(b, cc));
            if (mn < lo[c]) lo[c] = mn;
            if (mx > hi[c]) hi[c] = mx;
        }
        orc_v3 n = orc_cross(orc_mk(e1[3 * f], e1[3 * f + 1], e1[3 * f + 2]),
                             orc_mk(e2[3 * f], e2[3 * f + 1], e2[3 * f + 2]));
        double len = sqrt(orc_dot(n, n));
        nrm[3 * f] = n.x / len; nrm[3 * f + 1] = n.y / len; nrm[3 * f + 2] = n.z / len;
    }
    orc_stats st; memset(&st, 0, sizeof st);
    const orc_geom G = { v0, e1, e2, nrm, T, shininess };

    for (int jj = 0; jj < S; ++jj) {
        const uint32_t j = (uint32_t)(j0 + jj);
        /* O-step 1: photon travel direction s = -normalize(omega), basis (u, v). */
        orc_v3 om = orc_mk(sun_dirs[3 * jj], sun_dirs[3 * jj + 1], sun_dirs[3 * jj + 2]);
        orc_v3 s = orc_scale(orc_normalize(om), -1.0), bu, bv;
        orc_basis(s, &bu, &bv);
        /* O-step 2: emitter rectangle = projected AABB corners; photon weight. */
        double u0 = INFINITY, u1 = -INFINITY, vv0 = INFINITY, vv1 = -INFINITY, w0 = INFINITY;
        for (int c = 0; c < 8; ++c) {
            orc_v3 p = orc_mk((c & 1) ? hi[0] : lo[0], (c & 2) ? hi[1] : lo[1], (c & 4) ? hi[2] : lo[2]);
            double pu = orc_dot(p, bu), pv = orc_dot(p, bv), pw = orc_dot(p, s);
            u0 = fmin(u0, pu); u1 = fmax(u1, pu);
            vv0 = fmin(vv0, pv); vv1 = fmax(vv1, pv);
            w0 = fmin(w0, pw);
        }
        const double Ae = (u1 - u0) * (vv1 - vv0);
        const double wph = P * Ae / (double)N;
        double Fj[3] = { 0, 0, 0 }, Qj[3] = { 0, 0, 0 }, Tj[3] = { 0, 0, 0 }, TQj[3] = { 0, 0, 0 }, Dj[3] = { 0, 0, 0 };
        const orc_v3 xc = x_com ? orc_mk(x_com[0], x_com[1], x_com[2]) : orc_mk(0.0, 0.0, 0.0);

        for (long long i = 0; i < N && Ae > 0.0; ++i) {
            /* O-step 3: ray i. */
            uint32_t ctr[4] = { (uint32_t)i, j, (uint32_t)k, 0u }, r[4];
            orc_philox4x32_10(ctr, key, r);
            double pu, pv;
            if (opt->sampler == 0) {
                uint32_t cx, cy;
                deinterleave((uint64_t)i, &cx, &cy);
                pu = u0 + ((double)cx + orc_uniform(r[0])) / nx * (u1 - u0);
                pv = vv0 + ((double)cy + orc_uniform(r[1])) / ny * (vv1 - vv0);
            } else {
                pu = u0 + orc_uniform(r[0]) * (u1 - u0);
                pv = vv0 + orc_uniform(r[1]) * (vv1 - vv0);
            }
            orc_v3 o = orc_add(orc_add(orc_scale(bu, pu), orc_scale(bv, pv)), orc_scale(s, w0 - 1.0));
            orc_v3 d = s;
            double dp[3] = { 0, 0, 0 }, dq[3] = { 0, 0, 0 };
            unsigned long long sig = 0;
            st.launched++;
            trace_photon(&G, mats, o, d, -1, wph, (uint32_t)i, j, (uint32_t)k, 0u, key, opt, B, xc, &st, dp, dq,
                         first_hit ? &first_hit[(long long)jj * N + i] : NULL, &sig, F_direct ? Dj : NULL);
            for (int c = 0; c < 3; ++c) {
                Fj[c] += dp[c]; Qj[c] += dp[c] * dp[c];
                Tj[c] += dq[c]; TQj[c] += dq[c] * dq[c];
            }
            if (path_sig) path_sig[(long long)jj * N + i] = sig;
        }
        if (!(Ae > 0.0) && first_hit)
            for (long long i = 0; i < N; ++i) first_hit[(long long)jj * N + i] = -1;
        if (!(Ae > 0.0) && path_sig)
            for (long long i = 0; i < N; ++i) path_sig[(long long)jj * N + i] = 0;
        for (int c = 0; c < 3; ++c) {
            F[3 * jj + c] = Fj[c];
            if (sumsq) sumsq[3 * jj + c] = Qj[c];
            if (Tq) Tq[3 * jj + c] = Tj[c];
            if (tq_sumsq) tq_sumsq[3 * jj + c] = TQj[c];
            if (F_direct) F_direct[3 * jj + c] = Dj[c];
        }
    }
    if (stats) *stats = st;
    free(v0); free(e1); free(e2); free(nrm);
    return 0;
}

int srp_oracle_forces_torques_glossy(const float *verts, const float *mats, const float *shininess, long T, int k,
                              const float *sun_dirs, int S, int j0, long long N, int B,
                              unsigned long long seed, const orc_options *opt,
                              double *F, double *sumsq, orc_stats *stats, int *first_hit,
                              unsigned long long *path_sig, const double *x_com, double *Tq,
                              double *tq_sumsq)
{
    return forces_core(verts, mats, shininess, T, k, sun_dirs, S, j0, N, B, seed, opt, F, sumsq, stats, first_hit,
                       path_sig, x_com, Tq, tq_sumsq, NULL);
}

/* Total force and its direct part (depth-0 deposits); F_indirect = F - F_direct. */
int srp_oracle_forces_split(const float *verts, const float *mats, const float *shininess, long T, int k,
                            const float *sun_dirs, int S, int j0, long long N, int B, unsigned long long seed,
                            const orc_options *opt, double *F, double *F_direct, orc_stats *stats)
{
    if (!F_direct) return -1;
    return forces_core(verts, mats, shininess, T, k, sun_dirs, S, j0, N, B, seed, opt, F, NULL, stats, NULL, NULL,
                       NULL, NULL, NULL, F_direct);
}

/* Ideal-mirror specular lobes on every facet (R5): the call of the hot path. */
int srp_oracle_forces_torques(const float *verts, const float *mats, long T, int k,
                              const float *sun_dirs, int S, int j0, long long N, int B,
                              unsigned long long seed, const orc_options *opt,
                              double *F, double *sumsq, orc_stats *stats, int *first_hit,
                              unsigned long long *path_sig, const double *x_com, double *Tq,
                              double *tq_sumsq)
{
    return srp_oracle_forces_torques_glossy(verts, mats, NULL, T, k, sun_dirs, S, j0, N, B, seed, opt, F, sumsq,
                                            stats, first_hit, path_sig, x_com, Tq, tq_sumsq);
}

/* Forces only (the call the force tests and timings use). */
int srp_oracle_forces(const float *verts, const float *mats, long T, int k,
                      const float *sun_dirs, int S, int j0, long long N, int B,
                      unsigned long long seed, const orc_options *opt,
                      double *F, double *sumsq, orc_stats *stats, int *first_hit,
                      unsigned long long *path_sig)
{
    return srp_oracle_forces_torques(verts, mats, T, k, sun_dirs, S, j0, N, B, seed, opt, F, sumsq, stats,
                                     first_hit, path_sig, NULL, NULL, NULL);
}

/*
 * Thermal (local Lambertian) emitters, PAPER.md:606-612 (Sec. 5.9): "our simulation easily handles local sources
 * in the same way it does handle distant sun light ... we model thermal emission as Lambertian"; a Lambertian
 * emitter's momentum flux is 2/3 of a collimated beam's.  DESIGN.md reading R22.
 * Facet f of design k radiates |W_f| watts from the side of its normal n = normalize(e1 x e2) (W_f > 0) or of -n
 * (W_f < 0).  It launches N photons of momentum weight w = |W_f| / (c N) [newtons]: ray i draws
 * Philox(key = seed; ctr = (i, f, k, 0x80000000)) -> xi0..xi3; origin = uniform point of the triangle
 * x = v0 + sqrt(xi0) (1 - xi1) e1 + sqrt(xi0) xi1 e2; direction cosine-weighted about the emitting normal n_e in the
 * frame (t_u = e1/|e1|, t_v = n_e x t_u): phi = 2 pi xi2, rho = sqrt(xi3).  Recoil at emission: expected-value
 * deposit -(2/3) w n_e, analog deposit -w d, made at x.  The photon is then followed like any other (O-steps 4-7,
 * source triangle f excluded, lobe draws with counters (i, f, k, 0x80000000 | depth + 1)).
 * F double[3] (N), sumsq double[3] (per-photon totals squared, may be NULL), stats may be NULL.
 */
int srp_oracle_thermal_glossy(const float *verts, const float *mats, const float *shininess, long T, int k,
                              const float *facet_power, long long N, int B, unsigned long long seed,
                              const orc_options *opt, double *F, double *sumsq, orc_stats *stats)
{
    if (!verts || !mats || !facet_power || !F || !opt || T <= 0 || N <= 0 || B < 0 || B > 15) return -1;
    const double C_LIGHT = 299792458.0;
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    double *v0 = malloc(sizeof(double) * 3 * T), *e1 = malloc(sizeof(double) * 3 * T),
           *e2 = malloc(sizeof(double) * 3 * T), *nrm = malloc(sizeof(double) * 3 * T);
    for (long f = 0; f < T; ++f) {
        for (int c = 0; c < 3; ++c) {
            double a = verts[9 * f + c], b = verts[9 * f + 3 + c], cc = verts[9 * f + 6 + c];
            v0[3 * f + c] = a; e1[3 * f + c] = b - a; e2[3 * f + c] = cc - a;
        }
        orc_v3 n = orc_cross(orc_mk(e1[3 * f], e1[3 * f + 1], e1[3 * f + 2]),
                             orc_mk(e2[3 * f], e2[3 * f + 1], e2[3 * f + 2]));
        double len = sqrt(orc_dot(n, n));
        nrm[3 * f] = n.x / len; nrm[3 * f + 1] = n.y / len; nrm[3 * f + 2] = n.z / len;
    }
    const orc_geom G = { v0, e1, e2, nrm, T, shininess };
    orc_stats st; memset(&st, 0, sizeof st);
    double Ft[3] = { 0, 0, 0 }, Qt[3] = { 0, 0, 0 };
    const orc_v3 xc = orc_mk(0.0, 0.0, 0.0);
    for (long f = 0; f < T; ++f) {
        const double W = facet_power[f];
        if (W == 0.0) continue;
        const double w = fabs(W) / (C_LIGHT * (double)N);
        const orc_v3 E1 = orc_mk(e1[3 * f], e1[3 * f + 1], e1[3 * f + 2]), E2 = orc_mk(e2[3 * f], e2[3 * f + 1], e2[3 * f + 2]);
        const orc_v3 n = orc_mk(nrm[3 * f], nrm[3 * f + 1], nrm[3 * f + 2]);
        const orc_v3 ne = W > 0.0 ? n : orc_scale(n, -1.0);
        const orc_v3 tu = orc_normalize(E1), tv = orc_cross(ne, tu);
        for (long long i = 0; i < N; ++i) {
            uint32_t ctr[4] = { (uint32_t)i, (uint32_t)f, (uint32_t)k, 0x80000000u }, r[4];
            orc_philox4x32_10(ctr, key, r);
            const double x0 = orc_uniform(r[0]), x1 = orc_uniform(r[1]), x2 = orc_uniform(r[2]), x3 = orc_uniform(r[3]);
            const double su = sqrt(x0);
            const orc_v3 x = orc_add(orc_mk(v0[3 * f], v0[3 * f + 1], v0[3 * f + 2]),
                                     orc_add(orc_scale(E1, su * (1.0 - x1)), orc_scale(E2, su * x1)));
            const double phi = 6.283185307179586476925286766559 * x2, rho = sqrt(x3);
            const double lx = rho * cos(phi), ly = rho * sin(phi), lz = sqrt(1.0 - x3);
            const orc_v3 d = orc_add(orc_add(orc_scale(tu, lx), orc_scale(tv, ly)), orc_scale(ne, lz));
            double dp[3] = { 0, 0, 0 }, dq[3] = { 0, 0, 0 }, dd[3];
            if (opt->deposit == 0) { dd[0] = -(2.0 / 3.0) * w * ne.x; dd[1] = -(2.0 / 3.0) * w * ne.y; dd[2] = -(2.0 / 3.0) * w * ne.z; }
            else { dd[0] = -w * d.x; dd[1] = -w * d.y; dd[2] = -w * d.z; }
            orc_deposit(dd, x, xc, dp, dq);
            unsigned long long sig = 0;
            st.launched++;
            trace_photon(&G, mats, x, d, f, w, (uint32_t)i, (uint32_t)f, (uint32_t)k, 0x80000000u, key, opt, B, xc, &st,
                         dp, dq, NULL, &sig, NULL);
            for (int c = 0; c < 3; ++c) { Ft[c] += dp[c]; Qt[c] += dp[c] * dp[c]; }
        }
    }
    for (int c = 0; c < 3; ++c) { F[c] = Ft[c]; if (sumsq) sumsq[c] = Qt[c]; }
    if (stats) *stats = st;
    free(v0); free(e1); free(e2); free(nrm);
    return 0;
}

/*
 * The paper's own estimator, Eq. 5, backward from the surface -- a CROSS-CHECK of the forward
 * tracer above (reading R25), not a second product path:
 *   "a random triangle on the surface is chosen by sampling according to triangle area and a random point within
 *    that triangle using uniform point picking.  Next, we pick a random incoming direction and evaluate the radiation
 *    using a single sample of path tracing.  Finally, a random outgoing direction is selected ... We use BRDF
 *    importance sampling to generate the incoming and outgoing direction.  We also use next-event estimation ...
 *    at every light path vertex we check direct light from omega."
 * One sample i (Philox ctr (i, j, k, 0x40000000 | word)):
 *   1. facet f with probability A_f / A (inverse of the cumulative areas at xi0), x = v0 + sqrt(xi1)(1 - xi2) e1 +
 *      sqrt(xi1) xi2 e2.  Facets are two-sided (R6): both sides s = +n, -n are evaluated and added.
 *   2. direct light (next-event estimation at the first vertex): if n_s . w > 0 and the shadow ray x -> w (w = unit
 *      vector to the sun) is free, the side receives the pressure P cos(theta) along d = -w.
 *   3. indirect light: incoming direction w_in cosine-distributed about n_s (pdf cos/pi: the sampling density of a
 *      surface's response to light, which is proportional to <n, w_in>+ in Eq. 2); the radiance arriving along it is
 *      path-traced backwards from the surface point y the ray x + t w_in meets: at every vertex (at most B of them)
 *      direct sun light is added by next-event estimation through the Lambertian part rho_d / pi of the BRDF (a
 *      delta light cannot be seen through an ideal mirror), then the path goes on by BRDF importance sampling --
 *      absorbed with probability alpha, mirrored with rho_s, cosine-distributed with rho_d -- with throughput 1.
 *      With L in units of pressure per steradian the sample of step 3 is pi L received along d = -w_in.
 *   4. light received along d at x on side s deposits P_received [(alpha+rho_s+rho_d) d - rho_s r - 2/3 rho_d n_s]
 *      (expected value over the BRDF-sampled outgoing direction; opt->deposit = 1 draws w_out instead: nothing,
 *      the mirror direction, or a cosine-distributed one), sign per reading R1, times A (the pdf of step 1).
 * Equal in expectation to the forward tracer EXCEPT for sun light whose first reflection is specular: a backward
 * path ends at the sun only through next-event estimation, which an ideal mirror (a delta lobe, R3) never passes.
 * srp_oracle_forces with opt->no_caustics = 1 leaves exactly that light out.
 * F double[3], sumsq double[3] (squared per-sample totals; may be NULL), n_nee: shadow rays cast (may be NULL).
 */
static int blocked(const orc_geom *G, orc_v3 o, orc_v3 d, long src)
{
    double t;
    return closest_hit(G->v0, G->e1, G->e2, G->T, o, d, src, &t) >= 0;
}

static orc_v3 cosine_dir(const orc_geom *G, long f, orc_v3 nf, double u1, double u2)
{
    const double phi = 6.283185307179586476925286766559 * u1, rho = sqrt(u2);
    orc_v3 tu = orc_normalize(orc_mk(G->e1[3 * f], G->e1[3 * f + 1], G->e1[3 * f + 2]));
    orc_v3 tv = orc_cross(nf, tu);
    return orc_add(orc_add(orc_scale(tu, rho * cos(phi)), orc_scale(tv, rho * sin(phi))), orc_scale(nf, sqrt(1.0 - u2)));
}

int srp_oracle_backward(const float *verts, const float *mats, long T, int k, const float *sun_dir, int j,
                        long long N, int B, unsigned long long seed, const orc_options *opt,
                        double *F, double *sumsq, unsigned long long *n_nee)
{
    if (!verts || !mats || !sun_dir || !F || !opt || T <= 0 || N <= 0 || B < 0 || B > 15) return -1;
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    const double P = opt->solar_pressure;
    double *v0 = malloc(sizeof(double) * 3 * T), *e1 = malloc(sizeof(double) * 3 * T),
           *e2 = malloc(sizeof(double) * 3 * T), *nrm = malloc(sizeof(double) * 3 * T), *cum = malloc(sizeof(double) * T);
    double A = 0.0;
    for (long f = 0; f < T; ++f) {
        for (int c = 0; c < 3; ++c) {
            double a = verts[9 * f + c], b = verts[9 * f + 3 + c], cc = verts[9 * f + 6 + c];
            v0[3 * f + c] = a; e1[3 * f + c] = b - a; e2[3 * f + c] = cc - a;
        }
        orc_v3 n = orc_cross(orc_mk(e1[3 * f], e1[3 * f + 1], e1[3 * f + 2]), orc_mk(e2[3 * f], e2[3 * f + 1], e2[3 * f + 2]));
        double len = sqrt(orc_dot(n, n));
        nrm[3 * f] = n.x / len; nrm[3 * f + 1] = n.y / len; nrm[3 * f + 2] = n.z / len;
        A += 0.5 * len; cum[f] = A;
    }
    const orc_geom G = { v0, e1, e2, nrm, T, NULL };
    const orc_v3 w = orc_normalize(orc_mk(sun_dir[0], sun_dir[1], sun_dir[2]));
    double Ft[3] = { 0, 0, 0 }, Qt[3] = { 0, 0, 0 };
    unsigned long long nee = 0;
    for (long long i = 0; i < N; ++i) {
        uint32_t c0[4] = { (uint32_t)i, (uint32_t)j, (uint32_t)k, 0x40000000u }, r[4];
        orc_philox4x32_10(c0, key, r);
        /* step 1 */
        const double target = orc_uniform(r[0]) * A;
        long lo = 0, hi = T - 1;
        while (lo < hi) { long mid = (lo + hi) / 2; if (cum[mid] > target) hi = mid; else lo = mid + 1; }
        const long f = lo;
        const double su = sqrt(orc_uniform(r[1])), x2 = orc_uniform(r[2]);
        const orc_v3 E1 = orc_mk(e1[3 * f], e1[3 * f + 1], e1[3 * f + 2]), E2 = orc_mk(e2[3 * f], e2[3 * f + 1], e2[3 * f + 2]);
        const orc_v3 x = orc_add(orc_mk(v0[3 * f], v0[3 * f + 1], v0[3 * f + 2]),
                                 orc_add(orc_scale(E1, su * (1.0 - x2)), orc_scale(E2, su * x2)));
        const double al = mats[3 * f], rs = mats[3 * f + 1], rd = mats[3 * f + 2];
        double tot[3] = { 0, 0, 0 };
        for (int side = 0; side < 2; ++side) {
            const orc_v3 n = orc_mk(nrm[3 * f], nrm[3 * f + 1], nrm[3 * f + 2]);
            const orc_v3 ns = side == 0 ? n : orc_scale(n, -1.0);
            uint32_t c1[4] = { (uint32_t)i, (uint32_t)j, (uint32_t)k, 0x40000001u + (uint32_t)side }, q[4];
            orc_philox4x32_10(c1, key, q);
            /* light received at x on this side: up to two arrivals (direct, indirect), each "pressure along d" */
            orc_v3 dirs[2]; double press[2]; int n_arr = 0;
            /* step 2: direct light */
            const double cs = orc_dot(ns, w);
            if (cs > 0.0) {
                ++nee;
                if (!blocked(&G, x, w, f)) { dirs[n_arr] = orc_scale(w, -1.0); press[n_arr] = P * cs; ++n_arr; }
            }
            /* step 3: indirect light */
            if (B > 0) {
                const orc_v3 win = cosine_dir(&G, f, ns, orc_uniform(q[0]), orc_uniform(q[1]));
                orc_v3 o = x, dir = win; long src = f; double L = 0.0;
                for (int depth = 1; depth <= B; ++depth) {
                    double t;
                    const long g = closest_hit(G.v0, G.e1, G.e2, G.T, o, dir, src, &t);
                    if (g < 0) break;
                    const orc_v3 y = orc_add(o, orc_scale(dir, t));
                    orc_v3 ng = orc_mk(nrm[3 * g], nrm[3 * g + 1], nrm[3 * g + 2]);
                    if (orc_dot(ng, dir) > 0.0) ng = orc_scale(ng, -1.0);        /* the side the path arrives on */
                    const double cy = orc_dot(ng, w);
                    if (cy > 0.0) {
                        ++nee;
                        if (!blocked(&G, y, w, g)) L += (double)mats[3 * g + 2] / 3.14159265358979323846 * P * cy;
                    }
                    uint32_t c2[4] = { (uint32_t)i, (uint32_t)j, (uint32_t)k, 0x40000010u + 16u * (uint32_t)side + (uint32_t)depth }, z[4];
                    orc_philox4x32_10(c2, key, z);
                    const double z0 = orc_uniform(z[0]);
                    const float th1 = mats[3 * g], th2 = mats[3 * g] + mats[3 * g + 1];
                    if (z0 < (double)th1) break;                                  /* absorbed */
                    const orc_v3 wo = orc_scale(dir, -1.0);                      /* the direction the light leaves y in */
                    orc_v3 nd;
                    if (z0 < (double)th2) nd = orc_sub(orc_scale(ng, 2.0 * orc_dot(ng, wo)), wo);   /* mirror */
                    else nd = cosine_dir(&G, g, ng, orc_uniform(z[1]), orc_uniform(z[2]));
                    o = y; dir = nd; src = g;
                }
                if (L > 0.0) { dirs[n_arr] = orc_scale(win, -1.0); press[n_arr] = 3.14159265358979323846 * L; ++n_arr; }
            }
            /* step 4: force of what arrived */
            for (int a = 0; a < n_arr; ++a) {
                const orc_v3 d = dirs[a];
                const double cost = -orc_dot(d, ns);
                const orc_v3 refl = orc_add(d, orc_scale(ns, 2.0 * cost));
                double dd[3];
                if (opt->deposit == 0) {
                    const double s3 = al + rs + rd;
                    dd[0] = s3 * d.x - rs * refl.x - (2.0 / 3.0) * rd * ns.x;
                    dd[1] = s3 * d.y - rs * refl.y - (2.0 / 3.0) * rd * ns.y;
                    dd[2] = s3 * d.z - rs * refl.z - (2.0 / 3.0) * rd * ns.z;
                } else {
                    const double z0 = orc_uniform(q[2 + (a & 1)]);
                    const float th1 = mats[3 * f], th2 = mats[3 * f] + mats[3 * f + 1];
                    orc_v3 wout = orc_mk(0, 0, 0);
                    if (z0 < (double)th1) wout = orc_mk(0, 0, 0);
                    else if (z0 < (double)th2) wout = refl;
                    else {
                        uint32_t c3[4] = { (uint32_t)i, (uint32_t)j, (uint32_t)k, 0x40000004u + 2u * (uint32_t)side + (uint32_t)a }, u[4];
                        orc_philox4x32_10(c3, key, u);
                        wout = cosine_dir(&G, f, ns, orc_uniform(u[0]), orc_uniform(u[1]));
                    }
                    dd[0] = d.x - wout.x; dd[1] = d.y - wout.y; dd[2] = d.z - wout.z;
                }
                for (int c = 0; c < 3; ++c) tot[c] += A * press[a] * dd[c];
            }
        }
        for (int c = 0; c < 3; ++c) { Ft[c] += tot[c]; Qt[c] += tot[c] * tot[c]; }
    }
    for (int c = 0; c < 3; ++c) { F[c] = Ft[c] / (double)N; if (sumsq) sumsq[c] = Qt[c]; }
    if (n_nee) *n_nee = nee;
    free(v0); free(e1); free(e2); free(nrm); free(cum);
    return 0;
}

/* Philox and the uniform map exposed for the known-answer tests. */
void srp_oracle_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    orc_philox4x32_10(ctr, key, out);
}
double srp_oracle_uniform(uint32_t x) { return orc_uniform(x); }

int srp_oracle_thermal(const float *verts, const float *mats, long T, int k, const float *facet_power,
                       long long N, int B, unsigned long long seed, const orc_options *opt,
                       double *F, double *sumsq, orc_stats *stats)
{
    return srp_oracle_thermal_glossy(verts, mats, NULL, T, k, facet_power, N, B, seed, opt, F, sumsq, stats);
}
