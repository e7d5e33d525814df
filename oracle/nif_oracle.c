/* nif_oracle.c -- CPU ORACLE for the deformation-aware neural intersection query.
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code with
 * the CUDA path under paper_2604_24666_b200/ and neither includes the other.
 *
 * Plain, slow, single-threaded C99, one ray at a time, written from the paper
 * (/root/reference/PAPER.md, cited as P:line) with the readings listed in DESIGN.md
 * section 3 (cited as R#).  No blocking, fusion or reordering beyond what is stated.
 *
 * Precision: the north star (BASELINE.json:5) fixes "fp32 CPU implementation".  Steps O4/O5
 * (ray-voxel intersection) follow an exact fp32 operation sequence because hit ids must be
 * bit-exact.  Steps O8-O10 decide cells/indices in fp32 and accumulate in `acc_t`, which is
 * float by default and double when compiled with -DNIFO_ACC_DOUBLE (second library used
 * only to bound the fp32 oracle's own rounding; tests/test_oracle_network.py).
 *
 * Compile: gcc -O2 -std=c99 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/__init__.py).
 * -ffp-contract=off matters: a*b+c must never silently become an fma; every fused
 * operation below is an explicit fmaf().
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"):
 *   O2/O7 deformation    : printed values (tests/golden/deform_worked.txt), identity pose,
 *                          inverse(forward(x)) = x
 *   O2x exact lattice    : binary128 evaluation == mpmath at 60 digits rounded to fp32; the fp64
 *                          fast path + fallback == the binary128 evaluation on every lattice point
 *   O4/O5 voxel hit      : slab closed form on the identity pose, reversed-ray invariant
 *   O6 nearest voxel     : BVH == brute force, bit-exact
 *   O8 encode            : hand-computed toy table (tests/golden/hash_toy.txt), constant and
 *                          affine tables, torch grid_sample on dense levels, numpy sin/cos
 *   O9 MLP               : torch fp64 linear+relu chain
 *   O9b fp16 activations : round_f16 == numpy float16 conversion; numpy float16 chain
 *   O10 decode           : closed forms / invariants
 *   O11 walk             : per-voxel enumeration, DDA row, telescoping sum; O11x: the literal exit-face walk of
 *                          P:51 visits the same voxel sequence (differences classified, tests/test_oracle_multi.py)
 *   end-to-end accuracy against a trained model: PARITY UNPINNED (no weights/objects exist).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef NIFO_ACC_DOUBLE
typedef double acc_t;
#define ACC_EXP exp
#define ACC_EXPM1 expm1
#define ACC_SQRT sqrt
#else
typedef float acc_t;
#define ACC_EXP expf
#define ACC_EXPM1 expm1f
#define ACC_SQRT sqrtf
#endif

#define NIFO_N_OUT 12
#define NIFO_FLAG_OCCLUSION_ONLY 1u
#define NIFO_FLAG_LATTICE_INVERSE 4u /* O7b: voxel-local trilinear inverse from the lattice instead of the closed form */
#define NIFO_FLAG_DIST_LOG 2u       /* O10b: ReLU + log-transformed distance head (R24) */
#define NIFO_FLAG_ACT_F16 8u        /* O9b: MLP input features and hidden activations rounded to fp16 (B:8) */

int nifo_acc_bytes(void) { return (int)sizeof(acc_t); }

/* ------------------------------------------------------------------------------------ */
/* O1/O2  Rest lattice and forward deformation ("apply parameterized deformation to  */
/* obtain deformed voxels"; formulas: BASELINE.json configs B:7-11, R7).         */
/* fp64 throughout, ONE rounding to fp32 per coordinate at the end.                        */
/* ------------------------------------------------------------------------------------ */
static void forward_f64(double theta_max, double k, const double p[3], double out[3])
{
    /* twist about +y: angle a = theta_max (y+1)/2  (B:7: theta(y) = 0.5 (y+1) for theta_max=1) */
    double x = p[0], y = p[1], z = p[2];
    double a = theta_max * (y + 1.0) / 2.0;
    double ca = cos(a), sa = sin(a);
    double tx = x * ca + z * sa;
    double ty = y;
    double tz = -x * sa + z * ca;
    /* bend about z with curvature k: circular arc of radius 1/k centred at (0, 1/k) (B:8).
       Cancellation-free form, continuous at k -> 0; |k| < 1e-6 is the identity (R7). */
    if (fabs(k) < 1e-6) {
        out[0] = tx; out[1] = ty; out[2] = tz;
    } else {
        double al = k * tx;
        double sh = sin(al / 2.0);
        out[0] = (1.0 - k * ty) * sin(al) / k;
        out[1] = ty * cos(al) + 2.0 * sh * sh / k;
        out[2] = tz;
    }
}

void nifo_forward_f64(double theta_max, double k, int64_t n, const double* p, double* out)
{
    for (int64_t i = 0; i < n; ++i) forward_f64(theta_max, k, p + 3 * i, out + 3 * i);
}

/* ------------------------------------------------------------------------------------ */
/* O2x  The deformed lattice is the CORRECTLY ROUNDED fp32 value of the real-valued closed    */
/* form (R7, R28): inputs are the fp64 rest coordinate (2i-nv)/nv (one fp64          */
/* division, exact for power-of-two nv) and the pose parameters theta_max, k (fp32, exact in   */
/* fp64); the formula of forward_f64 is then a real function of those, and the lattice entry    */
/* is RN_fp32 of its value.  Hit ids must be bit-exact between two implementations            */
/* (BASELINE.json:5), and a lattice entry that differs in its last bit can move a grazing ray    */
/* to another voxel, so "each side's fp64 libm, rounded once" (round 1) is not a definition:    */
/* two libms differ in the last fp64 bit about once in 1e7 values and that flips an fp32         */
/* rounding.  The definition written out: forward_q evaluates the same formula in binary128      */
/* (__float128, libquadmath sinq/cosq: 113-bit significand, error < 2^-100 here) and rounds      */
/* ONCE to fp32 (a zero result is stored as +0).  nifo_deform_lattice reaches the same result faster: it evaluates in fp64,      */
/* whose absolute error is far below NIFO_LATTICE_E for coordinates of magnitude < 8, and falls  */
/* back to forward_q only where the fp64 value lies within NIFO_LATTICE_E of a midpoint between  */
/* two adjacent fp32 numbers (where the fp64 error could change the rounding).  Pin:              */
/* tests/test_oracle_lattice.py compares it bit for bit with forward_q on every point, and        */
/* forward_q with mpmath at 60 digits.                                                            */
/* ------------------------------------------------------------------------------------ */
#include <quadmath.h>

static void forward_q(float theta_max_f, float k_f, const double p[3], __float128 out[3])
{
    __float128 theta_max = (__float128)theta_max_f, k = (__float128)k_f;
    __float128 x = (__float128)p[0], y = (__float128)p[1], z = (__float128)p[2];
    __float128 one = (__float128)1.0, two = (__float128)2.0;
    __float128 a = theta_max * (y + one) / two;
    __float128 ca = cosq(a), sa = sinq(a);
    __float128 tx = x * ca + z * sa;
    __float128 ty = y;
    __float128 tz = -x * sa + z * ca;
    if (fabs((double)k_f) < 1e-6) {
        out[0] = tx; out[1] = ty; out[2] = tz;
    } else {
        __float128 al = k * tx;
        __float128 sh = sinq(al / two);
        out[0] = (one - k * ty) * sinq(al) / k;
        out[1] = ty * cosq(al) + two * sh * sh / k;
        out[2] = tz;
    }
}

/* exposed for pins: the definition, n points -> n x 3 floats (binary128 evaluation, one rounding) */
void nifo_forward_exact_f32(float theta_max, float k, int64_t n, const double* p, float* out)
{
    for (int64_t i = 0; i < n; ++i) {
        __float128 q[3];
        forward_q(theta_max, k, p + 3 * i, q);
        for (int a = 0; a < 3; ++a) {
            out[3 * i + a] = (float)q[a];
            if (out[3 * i + a] == 0.0f) out[3 * i + a] = 0.0f;   /* +0, never -0 (R28) */
        }
    }
}

#define NIFO_LATTICE_E 9.094947017729282e-13      /* 2^-40: >= 1000 fp64 ulps of any |coordinate| < 8 */

/* 1 if rounding the fp64 value v (absolute error <= NIFO_LATTICE_E) to fp32 could go either way */
static int rounding_ambiguous(double v)
{
    float f = (float)v;
    if (!isfinite(f)) return 1;
    double lo = 0.5 * ((double)f + (double)nextafterf(f, -INFINITY));   /* midpoints to both neighbours: exact in fp64 */
    double hi = 0.5 * ((double)f + (double)nextafterf(f, INFINITY));
    return fabs(v - lo) <= NIFO_LATTICE_E || fabs(v - hi) <= NIFO_LATTICE_E;
}

/* lattice point (i,j,k), 0<=i,j,k<=nv, rest position ((2i-nv)/nv, ...) evaluated in fp64 (O1).
   Output index (i + (nv+1)(j + (nv+1)k))*3.  Returns through *n_exact (optional) how many points
   needed the binary128 evaluation. */
void nifo_deform_lattice_counted(int nv, float theta_max, float bend_k, float* lattice, int64_t* n_exact)
{
    int np1 = nv + 1;
    int64_t cnt = 0;
    for (int k = 0; k <= nv; ++k)
        for (int j = 0; j <= nv; ++j)
            for (int i = 0; i <= nv; ++i) {
                double p[3], q[3];
                p[0] = (2.0 * i - nv) / nv;
                p[1] = (2.0 * j - nv) / nv;
                p[2] = (2.0 * k - nv) / nv;
                forward_f64((double)theta_max, (double)bend_k, p, q);
                float* o = lattice + 3 * ((size_t)i + (size_t)np1 * ((size_t)j + (size_t)np1 * k));
                if (rounding_ambiguous(q[0]) || rounding_ambiguous(q[1]) || rounding_ambiguous(q[2])) {
                    __float128 e[3];
                    forward_q(theta_max, bend_k, p, e);
                    o[0] = (float)e[0]; o[1] = (float)e[1]; o[2] = (float)e[2];
                    ++cnt;
                } else {
                    o[0] = (float)q[0]; o[1] = (float)q[1]; o[2] = (float)q[2];
                }
                for (int a = 0; a < 3; ++a)
                    if (o[a] == 0.0f) o[a] = 0.0f;           /* a zero coordinate is stored as +0 (R28) */
            }
    if (n_exact) *n_exact = cnt;
}

void nifo_deform_lattice(int nv, float theta_max, float bend_k, float* lattice)
{
    nifo_deform_lattice_counted(nv, theta_max, bend_k, lattice, 0);
}

/* ------------------------------------------------------------------------------------ */
/* O7  Inverse deformation of a deformed-space point, fp32 ("every deformed-space    */
/* hit point is transformed back into rest space using the inverse deformation").          */
/* Composite inverse = twist^-1(bend^-1(P)).                                              */
/* ------------------------------------------------------------------------------------ */
static void inverse_f32(float theta_max, float k, const float P[3], float out[3])
{
    float X = P[0], Y = P[1], Z = P[2];
    float bx, by, bz;
    if (fabsf(k) < 1e-6f) {
        bx = X; by = Y; bz = Z;
    } else {
        /* dx = (1-ky) sin(al), dy = (1-ky) cos(al), r = 1-ky; y = (1-r)/k written without
           cancellation as (2Y - k(X^2+Y^2)) / (1+r). */
        float dx = k * X;
        float dy = 1.0f - k * Y;
        float r = sqrtf(dx * dx + dy * dy);
        bx = atan2f(dx, dy) / k;
        by = (2.0f * Y - k * (X * X + Y * Y)) / (1.0f + r);
        bz = Z;
    }
    float a = -theta_max * (by + 1.0f) / 2.0f;
    float ca = cosf(a), sa = sinf(a);
    out[0] = bx * ca + bz * sa;
    out[1] = by;
    out[2] = -bx * sa + bz * ca;
}

void nifo_inverse_f32(float theta_max, float k, int64_t n, const float* P, float* out)
{
    for (int64_t i = 0; i < n; ++i) inverse_f32(theta_max, k, P + 3 * i, out + 3 * i);
}

/* ------------------------------------------------------------------------------------ */
/* O7b  Voxel-local inverse for a deformation given only as a deformed corner lattice        */
/* ("user-specified deformation"; "within each voxel the deformation field is      */
/* approximately linear"; R27).  Inside voxel (ix,iy,iz) the deformation is taken to be the   */
/* trilinear interpolant of its 8 deformed corners q_c, c = dx + 2 dy + 4 dz:                 */
/*   T(u,v,w) = sum_c q_c * (dx?u:1-u)(dy?v:1-v)(dz?w:1-w),  (u,v,w) in [0,1]^3 the position  */
/* inside the rest voxel.  T(u,v,w) = P is solved by Newton's method from the voxel centre,   */
/* NIFO_NEWTON_ITERS iterations, 3x3 system by Cramer's rule, all in fp32 (a singular         */
/* Jacobian stops the iteration).  Rest point: (2 (i + u) - Nv) / Nv per axis.  Points on the  */
/* voxel's triangulated faces may land slightly outside [0,1]^3; no clamp here (the encoder    */
/* clamps the normalised point, R3).                                                          */
/* ------------------------------------------------------------------------------------ */
#define NIFO_NEWTON_ITERS 5

static void inverse_trilinear_f32(const float* lattice, int nv, int32_t id, const float P[3], float out[3])
{
    int ix = id % nv, iy = (id / nv) % nv, iz = id / (nv * nv);
    int cell[3] = { ix, iy, iz };
    size_t np1 = (size_t)nv + 1;
    float q[8][3];
    for (int c = 0; c < 8; ++c) {
        const float* p = lattice + 3 * ((size_t)(ix + (c & 1)) + np1 * ((size_t)(iy + ((c >> 1) & 1)) + np1 * (size_t)(iz + (c >> 2))));
        q[c][0] = p[0]; q[c][1] = p[1]; q[c][2] = p[2];
    }
    float u = 0.5f, v = 0.5f, w = 0.5f;
    for (int it = 0; it < NIFO_NEWTON_ITERS; ++it) {
        float T[3], Ju[3], Jv[3], Jw[3], r[3];
        for (int a = 0; a < 3; ++a) {
            float d00 = q[1][a] - q[0][a], d10 = q[3][a] - q[2][a], d01 = q[5][a] - q[4][a], d11 = q[7][a] - q[6][a];
            float c00 = q[0][a] + u * d00, c10 = q[2][a] + u * d10, c01 = q[4][a] + u * d01, c11 = q[6][a] + u * d11;
            float e0 = c10 - c00, e1 = c11 - c01;
            float c0 = c00 + v * e0, c1 = c01 + v * e1;
            T[a] = c0 + w * (c1 - c0);
            Jw[a] = c1 - c0;
            Jv[a] = e0 + w * (e1 - e0);
            float f0 = d00 + v * (d10 - d00), f1 = d01 + v * (d11 - d01);
            Ju[a] = f0 + w * (f1 - f0);
            r[a] = P[a] - T[a];
        }
        /* Cramer: det[Ju Jv Jw], and the same determinant with one column replaced by r */
        float cx = Jv[1] * Jw[2] - Jv[2] * Jw[1], cy = Jv[2] * Jw[0] - Jv[0] * Jw[2], cz = Jv[0] * Jw[1] - Jv[1] * Jw[0];
        float det = Ju[0] * cx + Ju[1] * cy + Ju[2] * cz;
        if (det == 0.0f) break;
        float du = (r[0] * cx + r[1] * cy + r[2] * cz) / det;
        float rx = r[1] * Jw[2] - r[2] * Jw[1], ry = r[2] * Jw[0] - r[0] * Jw[2], rz = r[0] * Jw[1] - r[1] * Jw[0];
        float dv = (Ju[0] * rx + Ju[1] * ry + Ju[2] * rz) / det;
        float sx = Jv[1] * r[2] - Jv[2] * r[1], sy = Jv[2] * r[0] - Jv[0] * r[2], sz = Jv[0] * r[1] - Jv[1] * r[0];
        float dw = (Ju[0] * sx + Ju[1] * sy + Ju[2] * sz) / det;
        u += du; v += dv; w += dw;
    }
    float uvw[3] = { u, v, w };
    for (int a = 0; a < 3; ++a) out[a] = (2.0f * ((float)cell[a] + uvw[a]) - (float)nv) / (float)nv;
}

/* exposed for pins: rest point of P[i] taken to lie in voxel id[i] */
void nifo_inverse_trilinear(const float* lattice, int nv, int64_t n, const int32_t* id, const float* P, float* out)
{
    for (int64_t i = 0; i < n; ++i) inverse_trilinear_f32(lattice, nv, id[i], P + 3 * i, out + 3 * i);
}

/* ------------------------------------------------------------------------------------ */
/* O4  Ray-triangle: Moeller-Trumbore, two-sided, on the infinite line, fp32 ARITHMETIC    */
/* CONTRACT (R9).  Every operation is one IEEE binary32 round-to-nearest-even    */
/* operation; fmaf() is the only fused operation; nothing else may be contracted.          */
/* ------------------------------------------------------------------------------------ */
typedef struct { float x, y, z; } v3;

static v3 v3sub(v3 a, v3 b) { v3 r; r.x = a.x - b.x; r.y = a.y - b.y; r.z = a.z - b.z; return r; }

static v3 v3cross(v3 p, v3 q)
{
    v3 r;
    r.x = fmaf(p.y, q.z, -(p.z * q.y));
    r.y = fmaf(p.z, q.x, -(p.x * q.z));
    r.z = fmaf(p.x, q.y, -(p.y * q.x));
    return r;
}

static float v3dot(v3 p, v3 q) { return fmaf(p.z, q.z, fmaf(p.y, q.y, p.x * q.x)); }

static int tri_hit(v3 o, v3 d, v3 v0, v3 v1, v3 v2, float* t)
{
    v3 e1 = v3sub(v1, v0);
    v3 e2 = v3sub(v2, v0);
    v3 pv = v3cross(d, e2);
    float det = v3dot(e1, pv);
    if (det == 0.0f) return 0;
    float inv = 1.0f / det;
    v3 sv = v3sub(o, v0);
    float u = v3dot(sv, pv) * inv;
    v3 qv = v3cross(sv, e1);
    float v = v3dot(d, qv) * inv;
    if (!((u >= 0.0f) && (v >= 0.0f) && (u + v <= 1.0f))) return 0;   /* NaN rejects */
    float tt = v3dot(e2, qv) * inv;
    if (!isfinite(tt)) return 0;
    *t = tt;
    return 1;
}

/* O4b  Ray-box slab interval, fp32 contract (R10).  inv = 1/d per axis (IEEE, so a
   zero component gives +-inf).  Rounding is monotone in the box coordinate (and the NaN rule
   below preserves that), so for nested boxes the intervals nest EXACTLY -- this is what makes culling with
   any hierarchy of enclosing boxes provably equal to brute force. */
static int slab(const float lo[3], const float hi[3], const float o[3], const float inv[3],
                float* bn, float* bf)
{
    float tmin = -INFINITY, tmax = INFINITY;
    for (int a = 0; a < 3; ++a) {
        float t0 = (lo[a] - o[a]) * inv[a];
        float t1 = (hi[a] - o[a]) * inv[a];
        float tn = fminf(t0, t1), tf = fmaxf(t0, t1);
        /* 0*inf = NaN: the ray runs inside a face plane of the box (d[a] == 0 and o[a] on the
           plane).  Faces are inclusive: the axis does not constrain the interval. */
        if (t0 != t0 || t1 != t1) { tn = -INFINITY; tf = INFINITY; }
        tmin = fmaxf(tmin, tn);
        tmax = fminf(tmax, tf);
    }
    if (!((tmin <= tmax) && (tmax >= 0.0f))) return 0;
    *bn = fmaxf(tmin, 0.0f);
    *bf = tmax;
    return 1;
}

static v3 lattice_pt(const float* lattice, int nv, int i, int j, int k)
{
    size_t np1 = (size_t)nv + 1;
    const float* p = lattice + 3 * ((size_t)i + np1 * ((size_t)j + np1 * (size_t)k));
    v3 r; r.x = p[0]; r.y = p[1]; r.z = p[2];
    return r;
}

static void voxel_aabb(const float* lattice, int nv, int ix, int iy, int iz, float lo[3], float hi[3])
{
    lo[0] = lo[1] = lo[2] = INFINITY;
    hi[0] = hi[1] = hi[2] = -INFINITY;
    for (int c = 0; c < 8; ++c) {
        v3 q = lattice_pt(lattice, nv, ix + (c & 1), iy + ((c >> 1) & 1), iz + (c >> 2));
        lo[0] = fminf(lo[0], q.x); hi[0] = fmaxf(hi[0], q.x);
        lo[1] = fminf(lo[1], q.y); hi[1] = fmaxf(hi[1], q.y);
        lo[2] = fminf(lo[2], q.z); hi[2] = fmaxf(hi[2], q.z);
    }
}

/* O3 + O5  One deformed voxel = its 8 lattice corners mapped forward, intersected as 12
   triangles (B:7).  For axis a and side s, with (b,c) the other two axes in cyclic order,
   q_uv = corner with offset s on a, u on b, v on c; triangles (q00,q10,q11), (q00,q11,q01).
   Result: entry/exit parameters of the straight ray inside the voxel ("entry and
   exit points of ray segment i within occupied voxel i in deformed space").
   t_in = clamp(max(t_lo, box_near), .., box_far), t_out likewise (R10, R11). */
static int voxel_hit(const float* lattice, int nv, int ix, int iy, int iz,
                     const float o[3], const float d[3], const float inv[3],
                     float* t_in, float* t_out)
{
    float lo[3], hi[3], bn, bf;
    voxel_aabb(lattice, nv, ix, iy, iz, lo, hi);
    if (!slab(lo, hi, o, inv, &bn, &bf)) return 0;
    v3 O, D; O.x = o[0]; O.y = o[1]; O.z = o[2]; D.x = d[0]; D.y = d[1]; D.z = d[2];
    int base[3]; base[0] = ix; base[1] = iy; base[2] = iz;
    int any = 0;
    float tlo = INFINITY, thi = -INFINITY;
    for (int a = 0; a < 3; ++a) {
        int b = (a + 1) % 3, c = (a + 2) % 3;
        for (int s = 0; s < 2; ++s) {
            v3 q[2][2];
            for (int u = 0; u < 2; ++u)
                for (int v = 0; v < 2; ++v) {
                    int idx[3];
                    idx[a] = base[a] + s; idx[b] = base[b] + u; idx[c] = base[c] + v;
                    q[u][v] = lattice_pt(lattice, nv, idx[0], idx[1], idx[2]);
                }
            float t;
            if (tri_hit(O, D, q[0][0], q[1][0], q[1][1], &t)) { any = 1; tlo = fminf(tlo, t); thi = fmaxf(thi, t); }
            if (tri_hit(O, D, q[0][0], q[1][1], q[0][1], &t)) { any = 1; tlo = fminf(tlo, t); thi = fmaxf(thi, t); }
        }
    }
    if (!any) return 0;
    if (!(thi >= 0.0f)) return 0;                 /* whole voxel behind the origin */
    float ti = fminf(fmaxf(tlo, bn), bf);          /* origin inside => t_lo < 0 => t_in = 0 (B:10) */
    float to = fmaxf(fminf(thi, bf), ti);
    *t_in = ti; *t_out = to;
    return 1;
}

static void ray_inv(const float d[3], float inv[3])
{
    inv[0] = 1.0f / d[0]; inv[1] = 1.0f / d[1]; inv[2] = 1.0f / d[2];
}

int nifo_voxel_hit(const float* lattice, int nv, int voxel_id, const float* o, const float* d,
                   float* t_in, float* t_out)
{
    float inv[3]; ray_inv(d, inv);
    int ix = voxel_id % nv, iy = (voxel_id / nv) % nv, iz = voxel_id / (nv * nv);
    return voxel_hit(lattice, nv, ix, iy, iz, o, d, inv, t_in, t_out);
}

/* ------------------------------------------------------------------------------------ */
/* O6  Nearest deformed voxel = arg-min over ALL occupied voxels of (t_in, id)            */
/* ("intersecting the ray with the occupied deformed voxels ... The first             */
/* intersection point defines the starting voxel"; ties -> lowest id, R12).  This brute    */
/* force IS the definition.                                                               */
/* ------------------------------------------------------------------------------------ */
void nifo_traverse_brute(int nv, const uint8_t* occ, const float* lattice, int64_t n,
                         const float* origin, const float* dir,
                         int32_t* vid, float* t_in, float* t_out)
{
    for (int64_t r = 0; r < n; ++r) {
        const float* o = origin + 3 * r; const float* d = dir + 3 * r;
        float inv[3]; ray_inv(d, inv);
        int32_t best = -1; float bti = INFINITY, bto = INFINITY;
        for (int iz = 0; iz < nv; ++iz)
            for (int iy = 0; iy < nv; ++iy)
                for (int ix = 0; ix < nv; ++ix) {
                    int32_t id = ix + nv * (iy + nv * iz);
                    if (!occ[id]) continue;
                    float ti, to;
                    if (voxel_hit(lattice, nv, ix, iy, iz, o, d, inv, &ti, &to) && ti < bti) {
                        best = id; bti = ti; bto = to;       /* ids ascend: ties keep the lower id */
                    }
                }
        vid[r] = best; t_in[r] = bti; t_out[r] = bto;
    }
}

/* `after_t`, `after_id`: only voxels whose (t_in, id) is lexicographically GREATER than
   (after_t, after_id) are candidates -- the successor query of the multi-voxel walk (O11).
   (-INFINITY, -1) = no bound = the plain first-hit query. */
static int after_bound(float ti, int32_t id, float after_t, int32_t after_id)
{
    return (ti > after_t) || (ti == after_t && id > after_id);
}

/* O11 (definition)  Successor of (after_t, after_id) in the ray's sequence of hit voxels ordered by
   (t_in, id): the voxel the walk of P:51 moves to next ("explicitly determining the voxel face
   through which a ray exits, which allows correct selection of neighboring voxels"); gaps of empty
   voxels are skipped because only occupied voxels are candidates.  Brute force. */
void nifo_next_voxel_brute(int nv, const uint8_t* occ, const float* lattice, int64_t n,
                           const float* origin, const float* dir, const float* after_t,
                           const int32_t* after_id, int32_t* vid, float* t_in, float* t_out)
{
    for (int64_t r = 0; r < n; ++r) {
        const float* o = origin + 3 * r; const float* d = dir + 3 * r;
        float inv[3]; ray_inv(d, inv);
        int32_t best = -1; float bti = INFINITY, bto = INFINITY;
        for (int iz = 0; iz < nv; ++iz)
            for (int iy = 0; iy < nv; ++iy)
                for (int ix = 0; ix < nv; ++ix) {
                    int32_t id = ix + nv * (iy + nv * iz);
                    if (!occ[id]) continue;
                    float ti, to;
                    if (voxel_hit(lattice, nv, ix, iy, iz, o, d, inv, &ti, &to) &&
                        after_bound(ti, id, after_t[r], after_id[r]) && ti < bti) {
                        best = id; bti = ti; bto = to;
                    }
                }
        vid[r] = best; t_in[r] = bti; t_out[r] = bto;
    }
}

/* ------------------------------------------------------------------------------------ */
/* O6 (large inputs)  The oracle's own "simple BVH": binary, median split on   */
/* the longest axis of the voxel-box centres, leaves of <= 4 voxels, node box = exact      */
/* min/max union of its voxels' AABBs.  Culling uses slab() on the node box, which by the   */
/* nesting argument at slab() never rejects a voxel that voxel_hit() accepts and never     */
/* reports a node entry later than a contained voxel's t_in.  Validated bit-exactly against */
/* nifo_traverse_brute in tests/test_oracle_traverse.py.                                   */
/* ------------------------------------------------------------------------------------ */
typedef struct {
    float lo[3], hi[3];
    int32_t left, right;      /* children, or -1 for a leaf              */
    int32_t first, count;     /* leaf: range in the permuted voxel list  */
} onode;

typedef struct {
    int nv;
    int32_t n_vox;
    int32_t* vox;             /* permuted occupied voxel ids */
    float* vlo; float* vhi;   /* per occupied voxel (indexed like vox) AABB */
    onode* nodes; int32_t n_nodes;
    const float* lattice;     /* borrowed */
} obvh;

static int g_axis; static const float* g_ctr;
static int cmp_centre(const void* a, const void* b)
{
    int32_t ia = *(const int32_t*)a, ib = *(const int32_t*)b;
    float ca = g_ctr[3 * (size_t)ia + g_axis], cb = g_ctr[3 * (size_t)ib + g_axis];
    if (ca < cb) return -1;
    if (ca > cb) return 1;
    return (ia > ib) - (ia < ib);
}

static int32_t obvh_build_rec(obvh* b, int32_t* order, const float* lo, const float* hi,
                              const float* ctr, int32_t first, int32_t count)
{
    int32_t me = b->n_nodes++;
    onode* nd = &b->nodes[me];
    float clo[3] = {INFINITY, INFINITY, INFINITY}, chi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int a = 0; a < 3; ++a) { nd->lo[a] = INFINITY; nd->hi[a] = -INFINITY; }
    for (int32_t i = first; i < first + count; ++i) {
        size_t v = (size_t)order[i];
        for (int a = 0; a < 3; ++a) {
            nd->lo[a] = fminf(nd->lo[a], lo[3 * v + a]);
            nd->hi[a] = fmaxf(nd->hi[a], hi[3 * v + a]);
            clo[a] = fminf(clo[a], ctr[3 * v + a]);
            chi[a] = fmaxf(chi[a], ctr[3 * v + a]);
        }
    }
    nd->first = first; nd->count = count; nd->left = nd->right = -1;
    if (count <= 4) return me;
    int axis = 0;
    if (chi[1] - clo[1] > chi[axis] - clo[axis]) axis = 1;
    if (chi[2] - clo[2] > chi[axis] - clo[axis]) axis = 2;
    g_axis = axis; g_ctr = ctr;
    qsort(order + first, (size_t)count, sizeof(int32_t), cmp_centre);
    int32_t half = count / 2;
    int32_t l = obvh_build_rec(b, order, lo, hi, ctr, first, half);
    int32_t r = obvh_build_rec(b, order, lo, hi, ctr, first + half, count - half);
    b->nodes[me].left = l; b->nodes[me].right = r;      /* b->nodes does not move: preallocated */
    return me;
}

void* nifo_bvh_build(int nv, const uint8_t* occ, const float* lattice)
{
    obvh* b = (obvh*)calloc(1, sizeof(obvh));
    b->nv = nv; b->lattice = lattice;
    size_t total = (size_t)nv * nv * nv;
    int32_t n = 0;
    for (size_t i = 0; i < total; ++i) n += occ[i] ? 1 : 0;
    b->n_vox = n;
    int32_t* ids = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    float* lo = (float*)malloc(sizeof(float) * 3 * (size_t)(n > 0 ? n : 1));
    float* hi = (float*)malloc(sizeof(float) * 3 * (size_t)(n > 0 ? n : 1));
    float* ctr = (float*)malloc(sizeof(float) * 3 * (size_t)(n > 0 ? n : 1));
    int32_t* order = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t m = 0;
    for (size_t i = 0; i < total; ++i) {
        if (!occ[i]) continue;
        int ix = (int)(i % nv), iy = (int)((i / nv) % nv), iz = (int)(i / ((size_t)nv * nv));
        ids[m] = (int32_t)i;
        voxel_aabb(lattice, nv, ix, iy, iz, lo + 3 * (size_t)m, hi + 3 * (size_t)m);
        for (int a = 0; a < 3; ++a) ctr[3 * (size_t)m + a] = 0.5f * (lo[3 * (size_t)m + a] + hi[3 * (size_t)m + a]);
        order[m] = m; ++m;
    }
    b->nodes = (onode*)malloc(sizeof(onode) * (size_t)(2 * n + 1));
    b->n_nodes = 0;
    if (n > 0) obvh_build_rec(b, order, lo, hi, ctr, 0, n);
    b->vox = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    for (int32_t i = 0; i < n; ++i) b->vox[i] = ids[order[i]];
    b->vlo = lo; b->vhi = hi;                 /* kept only for nifo_bvh_bounds */
    free(ids); free(ctr); free(order);
    return b;
}

void nifo_bvh_destroy(void* h)
{
    obvh* b = (obvh*)h;
    if (!b) return;
    free(b->vox); free(b->vlo); free(b->vhi); free(b->nodes); free(b);
}

int32_t nifo_bvh_num_voxels(const void* h) { return ((const obvh*)h)->n_vox; }

/* bounding box of the posed object = root box (used by the harness to place cameras) */
void nifo_bvh_bounds(const void* h, float lo[3], float hi[3])
{
    const obvh* b = (const obvh*)h;
    for (int a = 0; a < 3; ++a) {
        lo[a] = b->n_nodes ? b->nodes[0].lo[a] : 0.0f;
        hi[a] = b->n_nodes ? b->nodes[0].hi[a] : 0.0f;
    }
}

static void traverse_bvh_after(const obvh* b, const float* o, const float* d, float after_t, int32_t after_id,
                               int32_t* vid, float* t_in, float* t_out)
{
    float inv[3]; ray_inv(d, inv);
    int32_t best = -1; float bti = INFINITY, bto = INFINITY;
    int32_t stack[128]; float stack_t[128]; int sp = 0;
    int nv = b->nv;
    float bn, bf;
    if (b->n_nodes && slab(b->nodes[0].lo, b->nodes[0].hi, o, inv, &bn, &bf)) {
        stack[sp] = 0; stack_t[sp] = bn; ++sp;
    }
    while (sp > 0) {
        --sp;
        int32_t ni = stack[sp];
        if (stack_t[sp] > bti) continue;              /* strictly later: cannot win, even on a tie */
        const onode* nd = &b->nodes[ni];
        if (nd->left < 0) {
            for (int32_t i = nd->first; i < nd->first + nd->count; ++i) {
                int32_t id = b->vox[i];
                int ix = id % nv, iy = (id / nv) % nv, iz = id / (nv * nv);
                float ti, to;
                if (voxel_hit(b->lattice, nv, ix, iy, iz, o, d, inv, &ti, &to) &&
                    after_bound(ti, id, after_t, after_id)) {
                    if (ti < bti || (ti == bti && id < best)) { best = id; bti = ti; bto = to; }
                }
            }
            continue;
        }
        float ln, lf, rn, rf;
        int hl = slab(b->nodes[nd->left].lo, b->nodes[nd->left].hi, o, inv, &ln, &lf);
        int hr = slab(b->nodes[nd->right].lo, b->nodes[nd->right].hi, o, inv, &rn, &rf);
        if (hl && hr) {                                /* push the farther one first */
            if (ln <= rn) { stack[sp] = nd->right; stack_t[sp++] = rn; stack[sp] = nd->left; stack_t[sp++] = ln; }
            else          { stack[sp] = nd->left; stack_t[sp++] = ln; stack[sp] = nd->right; stack_t[sp++] = rn; }
        } else if (hl) { stack[sp] = nd->left; stack_t[sp++] = ln; }
        else if (hr)   { stack[sp] = nd->right; stack_t[sp++] = rn; }
    }
    *vid = best; *t_in = bti; *t_out = bto;
}

static void traverse_bvh_one(const obvh* b, const float* o, const float* d,
                             int32_t* vid, float* t_in, float* t_out)
{
    traverse_bvh_after(b, o, d, -INFINITY, -1, vid, t_in, t_out);
}

void nifo_next_voxel_bvh(const void* h, int64_t n, const float* origin, const float* dir,
                         const float* after_t, const int32_t* after_id, int32_t* vid, float* t_in, float* t_out)
{
    const obvh* b = (const obvh*)h;
    for (int64_t r = 0; r < n; ++r)
        traverse_bvh_after(b, origin + 3 * r, dir + 3 * r, after_t[r], after_id[r], vid + r, t_in + r, t_out + r);
}

void nifo_traverse_bvh(const void* h, int64_t n, const float* origin, const float* dir,
                       int32_t* vid, float* t_in, float* t_out)
{
    const obvh* b = (const obvh*)h;
    for (int64_t r = 0; r < n; ++r)
        traverse_bvh_one(b, origin + 3 * r, dir + 3 * r, vid + r, t_in + r, t_out + r);
}

/* ------------------------------------------------------------------------------------ */
/* O8  Composite encoding psi(x) = phi(gamma(x))  (Eq. 1).                       */
/* gamma(x) = [x, {sin(2^k x), cos(2^k x)}_{k<B}]  (no factor pi: Eq. 1 literal, R4).      */
/* "each query point is first expanded via positional encoding, and the resulting          */
/* frequency-modulated samples are independently processed by the multi-level hash grid    */
/* encoder. The encoded features are then flattened".  The S = 1+2B samples are     */
/* three-vectors (R2), mapped affinely to the grid's [0,1]^3 domain (R3).            */
/* ------------------------------------------------------------------------------------ */
typedef struct {
    int32_t pe_bands, levels, log2_T, feat;
    int32_t hidden_layers, width;
    const int32_t* level_res;                 /* N_l, L entries */
    int32_t enc_mode;                         /* 0: psi = phi(gamma(x)) (Eq. 1); 1: psi = [gamma(x), phi(x)] (O8b) */
} nifo_net_desc;

/* features per endpoint */
static int enc_per_endpoint(const nifo_net_desc* nd)
{
    if (nd->enc_mode == 1) return 3 + 6 * nd->pe_bands + nd->levels * nd->feat;
    return (1 + 2 * nd->pe_bands) * nd->levels * nd->feat;
}

/* samples: S x 3 floats. p_0 = x_n; p_{1+2k} = (sin(2^k x_n)+1)/2; p_{2+2k} = (cos(2^k x_n)+1)/2 */
void nifo_pe_samples(int bands, const float xn[3], float* samples)
{
    for (int a = 0; a < 3; ++a) samples[a] = xn[a];
    for (int k = 0; k < bands; ++k) {
        float f = ldexpf(1.0f, k);
        for (int a = 0; a < 3; ++a) {
            float arg = f * xn[a];
            samples[3 * (1 + 2 * k) + a] = (sinf(arg) + 1.0f) * 0.5f;
            samples[3 * (2 + 2 * k) + a] = (cosf(arg) + 1.0f) * 0.5f;
        }
    }
}

/* One level phi_l ("features are interpolated from neighboring grid vertices").
   pos = p * N; cell c = min(floor(pos), N-1); w = pos - c.  Vertex (i,j,k) index:
   dense i + (N+1)(j + (N+1)k) if (N+1)^3 <= T, else the spatial hash of [MESK22]:
   (i*1 xor j*2654435761 xor k*805459861) mod T in uint32 wrap-around arithmetic (R6).
   Corner order (dx,dy,dz) = 000,100,010,110,001,101,011,111; weight = prod(d ? w : 1-w). */
void nifo_level_lookup(int N, int log2_T, const float p[3], uint32_t idx[8], float w[8])
{
    uint32_t c[3]; float f[3];
    for (int a = 0; a < 3; ++a) {
        float pos = p[a] * (float)N;
        float fl = floorf(pos);
        if (fl > (float)(N - 1)) fl = (float)(N - 1);
        if (fl < 0.0f) fl = 0.0f;
        c[a] = (uint32_t)fl;
        f[a] = pos - fl;
    }
    uint64_t T = (uint64_t)1 << log2_T;
    uint64_t np1 = (uint64_t)N + 1;
    int dense = (np1 * np1 * np1 <= T);
    for (int corner = 0; corner < 8; ++corner) {
        int dx = corner & 1, dy = (corner >> 1) & 1, dz = corner >> 2;
        uint32_t i = c[0] + (uint32_t)dx, j = c[1] + (uint32_t)dy, k = c[2] + (uint32_t)dz;
        if (dense) idx[corner] = (uint32_t)(i + np1 * (j + np1 * k));
        else idx[corner] = ((i * 1u) ^ (j * 2654435761u) ^ (k * 805459861u)) & (uint32_t)(T - 1);
        float wx = dx ? f[0] : 1.0f - f[0];
        float wy = dy ? f[1] : 1.0f - f[1];
        float wz = dz ? f[2] : 1.0f - f[2];
        w[corner] = (wx * wy) * wz;
    }
}

/* psi for ONE endpoint: out[(s*L + l)*F + f].  table[l][index][f], every level T entries. */
static void encode_point(const nifo_net_desc* nd, const float* table, const float xn[3], acc_t* out)
{
    int S = 1 + 2 * nd->pe_bands, L = nd->levels, F = nd->feat;
    size_t T = (size_t)1 << nd->log2_T;
    float samples[3 * 64];
    if (nd->enc_mode == 1) {
        /* O8b  Concatenation reading of the hybrid encoding (B:5 "positional frequency terms plus a
           multiresolution hash grid"; R1 alternative): psi(x) = [ x, sin(2^0 x), cos(2^0 x), ...,
           sin(2^(B-1) x), cos(2^(B-1) x), phi(x) ] -- gamma(x) of P:75 handed to the MLP as it is
           (3 + 6B scalars, per band sin of the three axes then cos of the three axes, no pi: R4),
           followed by the grid features of the point itself, out[3 + 6B + l*F + f]. */
        for (int a = 0; a < 3; ++a) out[a] = (acc_t)xn[a];
        for (int k = 0; k < nd->pe_bands; ++k) {
            float f = ldexpf(1.0f, k);
            for (int a = 0; a < 3; ++a) {
                float arg = f * xn[a];
                out[3 + 6 * k + a] = (acc_t)sinf(arg);
                out[3 + 6 * k + 3 + a] = (acc_t)cosf(arg);
            }
        }
        out += 3 + 6 * nd->pe_bands;
        S = 1;
        for (int a = 0; a < 3; ++a) samples[a] = xn[a];
    } else {
        nifo_pe_samples(nd->pe_bands, xn, samples);
    }
    for (int s = 0; s < S; ++s)
        for (int l = 0; l < L; ++l) {
            uint32_t idx[8]; float w[8];
            nifo_level_lookup(nd->level_res[l], nd->log2_T, samples + 3 * s, idx, w);
            const float* lvl = table + (size_t)l * T * F;
            for (int f = 0; f < F; ++f) {
                acc_t acc = 0;
                for (int c = 0; c < 8; ++c) acc += (acc_t)w[c] * (acc_t)lvl[(size_t)idx[c] * F + f];
                out[((size_t)s * L + l) * F + f] = acc;
            }
        }
}

/* exposed for pins: features of n points (each an already normalised x_n), float output */
void nifo_encode(const nifo_net_desc* nd, const float* table, int64_t n, const float* xn, float* out)
{
    int per = enc_per_endpoint(nd);
    acc_t* tmp = (acc_t*)malloc(sizeof(acc_t) * (size_t)per);
    for (int64_t i = 0; i < n; ++i) {
        encode_point(nd, table, xn + 3 * i, tmp);
        for (int j = 0; j < per; ++j) out[(size_t)i * per + j] = (float)tmp[j];
    }
    free(tmp);
}

/* ------------------------------------------------------------------------------------ */
/* O9  MLP ("The retrieved grid features are concatenated and passed to a multi-layer */
/* perceptron").  a0 = input; a_i = ReLU(W_i a_{i-1}), i=1..H; z = W_{H+1} a_H.  No biases, */
/* linear output (R16).  weights[i]: row-major (fan_out, fan_in).                          */
/* ------------------------------------------------------------------------------------ */
/* O9b  BASELINE.json config 1 (B:8) fixes the precision of the fp16 networks: "fp16 weights and
   activations, fp32 accumulate".  round_f16 is IEEE binary16 round-to-nearest-even of one value
   (11-bit significand: quantum 2^(e-10) in the binade 2^e, fixed quantum 2^-24 below 2^-14,
   overflow above 65504 to infinity), returned as a float.  With act_f16 the MLP input features and
   every hidden activation (after ReLU) are rounded that way; products and sums stay in acc_t.  The
   default (act_f16 = 0) keeps activations in acc_t: the "fp32 oracle" of the north star.  The
   rounded mode exists because an argmax is an integer decided by floating point, and such a decision
   is to be taken in the same precision on both sides (the material argmax gate of DESIGN.md 3).
   Pin: tests/test_oracle_network.py compares round_f16 with numpy's float16 conversion. */
static float round_f16(float v)
{
    if (!(fabsf(v) < INFINITY) || v == 0.0f) return v;      /* inf, NaN, +-0 */
    int e;
    (void)frexpf(v, &e);                                    /* |v| = m 2^e, m in [0.5, 1) */
    int q = e - 11;                                         /* quantum exponent */
    if (q < -24) q = -24;
    float r = ldexpf(nearbyintf(ldexpf(v, -q)), q);         /* default rounding mode: ties to even */
    if (fabsf(r) > 65504.0f) r = copysignf(INFINITY, v);
    return r;
}

void nifo_round_f16(int64_t n, const float* in, float* out)
{
    for (int64_t i = 0; i < n; ++i) out[i] = round_f16(in[i]);
}

static void mlp_forward(const nifo_net_desc* nd, const float* const* weights, int d_in,
                        const acc_t* input, int n_out, acc_t* z, acc_t* buf0, acc_t* buf1, int act_f16)
{
    const acc_t* cur = input; int cur_n = d_in;
    acc_t* bufs[2] = { buf0, buf1 };
    for (int layer = 0; layer < nd->hidden_layers; ++layer) {
        acc_t* nxt = bufs[layer & 1];
        const float* W = weights[layer];
        for (int o = 0; o < nd->width; ++o) {
            acc_t acc = 0;
            for (int k = 0; k < cur_n; ++k) acc += (acc_t)W[(size_t)o * cur_n + k] * cur[k];
            nxt[o] = acc > 0 ? acc : 0;
            if (act_f16) nxt[o] = (acc_t)round_f16((float)nxt[o]);
        }
        cur = nxt; cur_n = nd->width;
    }
    const float* W = weights[nd->hidden_layers];
    for (int o = 0; o < n_out; ++o) {
        acc_t acc = 0;
        for (int k = 0; k < cur_n; ++k) acc += (acc_t)W[(size_t)o * cur_n + k] * cur[k];
        z[o] = acc;
    }
}

/* exposed for pins: n inputs of length d_in -> n x 12 logits */
void nifo_mlp(const nifo_net_desc* nd, const float* const* weights, int d_in, int64_t n,
              const float* input, float* logits)
{
    acc_t* in = (acc_t*)malloc(sizeof(acc_t) * (size_t)d_in);
    acc_t* b0 = (acc_t*)malloc(sizeof(acc_t) * (size_t)nd->width);
    acc_t* b1 = (acc_t*)malloc(sizeof(acc_t) * (size_t)nd->width);
    for (int64_t i = 0; i < n; ++i) {
        acc_t z[NIFO_N_OUT];
        for (int j = 0; j < d_in; ++j) in[j] = (acc_t)input[(size_t)i * d_in + j];
        mlp_forward(nd, weights, d_in, in, NIFO_N_OUT, z, b0, b1, 0);
        for (int j = 0; j < NIFO_N_OUT; ++j) logits[(size_t)i * NIFO_N_OUT + j] = (float)z[j];
    }
    free(in); free(b0); free(b1);
}

/* ------------------------------------------------------------------------------------ */
/* O10  Heads (order and activations B:7): occlusion sigma(z0); distance        */
/* d = sigma(z1) * l with l = t_out - t_in ("local hit distance t_i in [0, l_i] is      */
/* measured from the segment entry point"); D = t_in + d (P:61 with k = 0, delta_0 = t_in,   */
/* R13); normal = z2..4 / sqrt(max(z.z, 1e-24)); albedo sigma(z5..7); material logits z8..11. */
/* ------------------------------------------------------------------------------------ */
static acc_t sigmoid_acc(acc_t z) { return (acc_t)1 / ((acc_t)1 + ACC_EXP(-z)); }

void nifo_decode(int64_t n, const float* logits, const float* t_in, const float* t_out,
                 float* occlusion, float* distance, float* dist_total,
                 float* normal, float* albedo, float* material)
{
    for (int64_t i = 0; i < n; ++i) {
        const float* z = logits + NIFO_N_OUT * i;
        acc_t ell = (acc_t)(t_out[i] - t_in[i]);
        acc_t s = sigmoid_acc((acc_t)z[1]);
        acc_t d = s * ell;
        occlusion[i] = (float)sigmoid_acc((acc_t)z[0]);
        distance[i] = (float)d;
        dist_total[i] = (float)((acc_t)t_in[i] + d);
        acc_t nn = (acc_t)z[2] * z[2] + (acc_t)z[3] * z[3] + (acc_t)z[4] * z[4];
        acc_t inv = (acc_t)1 / ACC_SQRT(nn > (acc_t)1e-24 ? nn : (acc_t)1e-24);
        for (int a = 0; a < 3; ++a) {
            normal[3 * i + a] = (float)((acc_t)z[2 + a] * inv);
            albedo[3 * i + a] = (float)sigmoid_acc((acc_t)z[5 + a]);
        }
        for (int a = 0; a < 4; ++a) material[4 * i + a] = z[8 + a];
    }
}

/* ------------------------------------------------------------------------------------ */
/* Whole query, one ray at a time (Fig. 2): nearest deformed voxel -> entry/exit   */
/* points -> inverse deformation -> normalise to [0,1]^3 -> psi(entry) ++ psi(exit) (B:7)   */
/* -> MLP -> heads.  Miss: id -1, t = +inf, every network output 0 (R18).                  */
/* `bvh` may be NULL: then the brute-force definition is used.                             */
/* Network outputs may be NULL to run traversal only.                                      */
/* ------------------------------------------------------------------------------------ */
/* O7-O10 for ONE ray whose voxel (id, ti, to) is known: entry/exit points -> inverse deformation ->
   normalise -> psi(entry) ++ psi(exit) -> MLP -> heads, written to the pointers given (each
   pointing at this ray's slot; optional ones may be NULL). */
static void nifo_eval_voxel(const float* lattice, int nv, float theta_max, float bend_k, const nifo_net_desc* nd, const float* table,
                            const float* const* weights, const float* o, const float* d, uint32_t flags,
                            int32_t id, float ti, float to,
                            int32_t* vid, float* t_in, float* t_out,
                            float* occlusion, float* distance, float* dist_total,
                            float* normal, float* albedo, float* material, float* raw_logits)
{
    int per = enc_per_endpoint(nd), d_in = 2 * per;
    int n_out = (flags & NIFO_FLAG_OCCLUSION_ONLY) ? 1 : NIFO_N_OUT;
    acc_t* in = (acc_t*)malloc(sizeof(acc_t) * (size_t)d_in);
    acc_t* b0 = (acc_t*)malloc(sizeof(acc_t) * (size_t)nd->width);
    acc_t* b1 = (acc_t*)malloc(sizeof(acc_t) * (size_t)nd->width);
    *vid = id; *t_in = ti; *t_out = to;
    /* O7: P = o + t d as one fma per coordinate, inverse deformation, normalise */
    for (int e = 0; e < 2; ++e) {
        float t = e ? to : ti;
        float P[3], pr[3], xn[3];
        for (int a = 0; a < 3; ++a) P[a] = fmaf(t, d[a], o[a]);
        if (flags & NIFO_FLAG_LATTICE_INVERSE) inverse_trilinear_f32(lattice, nv, id, P, pr);
        else inverse_f32(theta_max, bend_k, P, pr);
        for (int a = 0; a < 3; ++a) {
            float v = (pr[a] + 1.0f) * 0.5f;
            xn[a] = v < 0.0f ? 0.0f : (v > 1.0f ? 1.0f : v);
        }
        encode_point(nd, table, xn, in + (size_t)e * per);
    }
    acc_t z[NIFO_N_OUT];
    float zf[NIFO_N_OUT];
    for (int j = 0; j < NIFO_N_OUT; ++j) z[j] = 0;
    if (flags & NIFO_FLAG_ACT_F16)
        for (int j = 0; j < d_in; ++j) in[j] = (acc_t)round_f16((float)in[j]);
    mlp_forward(nd, weights, d_in, in, n_out, z, b0, b1, (flags & NIFO_FLAG_ACT_F16) != 0);
    for (int j = 0; j < NIFO_N_OUT; ++j) zf[j] = (float)z[j];
    if (raw_logits) for (int j = 0; j < NIFO_N_OUT; ++j) raw_logits[j] = zf[j];
    if (flags & NIFO_FLAG_OCCLUSION_ONLY) {
        *occlusion = (float)sigmoid_acc(z[0]);
    } else {
        /* decode from the acc_t logits (not the float copies) */
        acc_t ell = (acc_t)(to - ti);
        *occlusion = (float)sigmoid_acc(z[0]);
        if (flags & NIFO_FLAG_DIST_LOG) {
            /* O10b ("We replace the sigmoid output with ReLU and regress log-transformed distances";
               R24): y = ReLU(z1) is the log-transformed ACCUMULATED distance, y = log(1 + D), so
               D = exp(y) - 1 >= 0; the part inside the voxel is D - t_in. */
            acc_t y = z[1] > (acc_t)0 ? z[1] : (acc_t)0;
            acc_t D = ACC_EXPM1(y);
            *dist_total = (float)D;
            *distance = (float)(D - (acc_t)ti);
        } else {
            acc_t s = sigmoid_acc(z[1]);
            acc_t dd = s * ell;
            *distance = (float)dd;
            *dist_total = (float)((acc_t)ti + dd);
        }
        acc_t nn = z[2] * z[2] + z[3] * z[3] + z[4] * z[4];
        acc_t inv = (acc_t)1 / ACC_SQRT(nn > (acc_t)1e-24 ? nn : (acc_t)1e-24);
        for (int a = 0; a < 3; ++a) {
            normal[a] = (float)(z[2 + a] * inv);
            albedo[a] = (float)sigmoid_acc(z[5 + a]);
        }
        for (int a = 0; a < 4; ++a) material[a] = zf[8 + a];
    }
    free(in); free(b0); free(b1);
}

int nifo_query(int nv, const uint8_t* occ, const float* lattice, const void* bvh,
               float theta_max, float bend_k,
               const nifo_net_desc* nd, const float* table, const float* const* weights,
               int64_t n, const float* origin, const float* dir, uint32_t flags,
               int32_t* vid, float* t_in, float* t_out,
               float* occlusion, float* distance, float* dist_total,
               float* normal, float* albedo, float* material, float* raw_logits)
{
    if (1 + 2 * nd->pe_bands > 64) return -1;
    for (int64_t r = 0; r < n; ++r) {
        const float* o = origin + 3 * r; const float* d = dir + 3 * r;
        if (bvh) traverse_bvh_one((const obvh*)bvh, o, d, vid + r, t_in + r, t_out + r);
        else nifo_traverse_brute(nv, occ, lattice, 1, o, d, vid + r, t_in + r, t_out + r);
        if (!occlusion) continue;
        if (vid[r] < 0) {
            occlusion[r] = 0.0f;
            if (distance) { distance[r] = 0.0f; dist_total[r] = 0.0f; }
            if (normal) for (int a = 0; a < 3; ++a) { normal[3 * r + a] = 0.0f; albedo[3 * r + a] = 0.0f; }
            if (material) for (int a = 0; a < 4; ++a) material[4 * r + a] = 0.0f;
            if (raw_logits) for (int j = 0; j < NIFO_N_OUT; ++j) raw_logits[NIFO_N_OUT * r + j] = 0.0f;
            continue;
        }
        nifo_eval_voxel(lattice, nv, theta_max, bend_k, nd, table, weights, o, d, flags, vid[r], t_in[r], t_out[r],
                        vid + r, t_in + r, t_out + r, occlusion + r, distance ? distance + r : 0,
                        dist_total ? dist_total + r : 0, normal ? normal + 3 * r : 0, albedo ? albedo + 3 * r : 0,
                        material ? material + 4 * r : 0, raw_logits ? raw_logits + NIFO_N_OUT * r : 0);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* O11x  The voxel walk as P:51 words it, literally: "we adopt a geometry-aware traversal by    */
/* explicitly determining the voxel face through which a ray exits, which allows correct         */
/* selection of neighboring voxels"; the first voxel comes from the BVH.  This is a PIN    */
/* for reading R22 (the product and O11 define the walk as the successor in (t_in, id) order      */
/* over all occupied voxels), not a product path.  One ray: start in the first occupied voxel     */
/* (O6).  In the current lattice cell (occupied or not -- every cell of the lattice has its 8      */
/* deformed corners) intersect the ray with the cell's 12 triangles (O3/O4); the accepted          */
/* intersection with the largest t is where the ray leaves the cell and the face that triangle     */
/* lies on is the exit face (axis a, side s); the next cell is the lattice neighbour across it.     */
/* Unoccupied cells are stepped through the same way; leaving the grid ends the walk.  `seq`        */
/* receives the occupied cells in the order they are entered (the first voxel included).           */
/* status: 0 = left the grid; 1 = no progress (the cell is only touched: exit t <= the t at which  */
/* it was entered -- a ray through an edge or corner, where "the exit face" is not defined);        */
/* 2 = no triangle of the cell accepted the ray; 3 = max_vox occupied voxels recorded; -1 = the    */
/* ray hits no occupied voxel at all.                                                              */
/* ------------------------------------------------------------------------------------ */
static int cell_exit_face(const float* lattice, int nv, const int cell[3], v3 O, v3 D, int* axis, int* side, float* t_exit)
{
    int any = 0; float best = -INFINITY;
    for (int a = 0; a < 3; ++a) {
        int b = (a + 1) % 3, c = (a + 2) % 3;
        for (int s = 0; s < 2; ++s) {
            v3 q[2][2];
            for (int u = 0; u < 2; ++u)
                for (int v = 0; v < 2; ++v) {
                    int idx[3];
                    idx[a] = cell[a] + s; idx[b] = cell[b] + u; idx[c] = cell[c] + v;
                    q[u][v] = lattice_pt(lattice, nv, idx[0], idx[1], idx[2]);
                }
            float t;
            if (tri_hit(O, D, q[0][0], q[1][0], q[1][1], &t) && (!any || t > best)) { any = 1; best = t; *axis = a; *side = s; }
            if (tri_hit(O, D, q[0][0], q[1][1], q[0][1], &t) && (!any || t > best)) { any = 1; best = t; *axis = a; *side = s; }
        }
    }
    *t_exit = best;
    return any;
}

void nifo_exit_face_walk(int nv, const uint8_t* occ, const float* lattice, const void* bvh,
                         int64_t n, const float* origin, const float* dir, int max_vox,
                         int32_t* seq, int32_t* status)
{
    for (int64_t r = 0; r < n; ++r) {
        const float* o = origin + 3 * r; const float* d = dir + 3 * r;
        int32_t* out = seq + (size_t)r * max_vox;
        for (int k = 0; k < max_vox; ++k) out[k] = -1;
        int32_t id; float ti, to;
        if (bvh) traverse_bvh_one((const obvh*)bvh, o, d, &id, &ti, &to);
        else nifo_traverse_brute(nv, occ, lattice, 1, o, d, &id, &ti, &to);
        if (id < 0) { status[r] = -1; continue; }
        v3 O, D; O.x = o[0]; O.y = o[1]; O.z = o[2]; D.x = d[0]; D.y = d[1]; D.z = d[2];
        int cell[3]; cell[0] = id % nv; cell[1] = (id / nv) % nv; cell[2] = id / (nv * nv);
        int count = 0;
        out[count++] = id;
        float t_entered = -INFINITY;
        int st = 0;
        for (;;) {
            int axis = 0, side = 0; float t_exit;
            if (!cell_exit_face(lattice, nv, cell, O, D, &axis, &side, &t_exit)) { st = 2; break; }
            if (!(t_exit > t_entered)) { st = 1; break; }
            cell[axis] += side ? 1 : -1;
            if (cell[axis] < 0 || cell[axis] >= nv) { st = 0; break; }
            t_entered = t_exit;
            int32_t nid = cell[0] + nv * (cell[1] + nv * cell[2]);
            if (occ[nid]) {
                if (count == max_vox) { st = 3; break; }
                out[count++] = nid;
            }
        }
        status[r] = st;
    }
}

/* ------------------------------------------------------------------------------------ */
/* O11  Multi-voxel walk at evaluation time (P:51 voxel traversal under deformation, P:53 BVH   */
/* start, P:59-61 segmented distance, "During evaluation, we reconstruct hit positions     */
/* along the same segmented ray").  For one ray: visit the occupied voxels it crosses in order   */
/* of (t_in, id); evaluate the network on each voxel's rest-space segment; stop at the first     */
/* voxel k whose predicted occlusion is >= 0.5 (logit z0 >= 0; R22).  Distance:        */
/* D = sum_{j<k}(delta_j + l_j) + delta_k + t_k accumulated segment by segment along the */
/* ray, with x_{-1}^1 := ray origin (R13), t_k = sigmoid(z1) * l_k (R14), l_j = t_out,j - t_in,j */
/* and the gap delta_j = t_in,j - t_out,j-1 taken SIGNED (R23): P:59 defines it as a norm, which */
/* is the same number whenever consecutive segments do not overlap; warped voxels can overlap    */
/* along the ray, and a norm would then count the overlap twice.  status: 1 = hit accepted at voxel k, 0 = the ray left the     */
/* object without a predicted hit (outputs as for a miss, R18), 2 = max_steps voxels evaluated   */
/* without a hit (outputs of the last voxel evaluated).  steps = voxels evaluated.               */
/* ------------------------------------------------------------------------------------ */
int nifo_query_multi(int nv, const uint8_t* occ, const float* lattice, const void* bvh,
                     float theta_max, float bend_k,
                     const nifo_net_desc* nd, const float* table, const float* const* weights,
                     int64_t n, const float* origin, const float* dir, uint32_t flags, int max_steps,
                     int32_t* vid, float* t_in, float* t_out,
                     float* occlusion, float* distance, float* dist_total,
                     float* normal, float* albedo, float* material, float* raw_logits,
                     int32_t* status, int32_t* steps, float* dist_accum)
{
    for (int64_t r = 0; r < n; ++r) {
        const float* o = origin + 3 * r; const float* d = dir + 3 * r;
        float after_t = -INFINITY; int32_t after_id = -1;
        float prev_exit = 0.0f;                              /* x_{-1}^1 := ray origin (R13): parameter 0 */
        float acc = 0.0f;                                    /* sum_{j<k} (delta_j + l_j) */
        int32_t st = 0, k = 0;
        for (;;) {
            int32_t id; float ti, to;
            if (bvh) traverse_bvh_after((const obvh*)bvh, o, d, after_t, after_id, &id, &ti, &to);
            else nifo_next_voxel_brute(nv, occ, lattice, 1, o, d, &after_t, &after_id, &id, &ti, &to);
            if (id < 0) {                                    /* left the object: miss outputs */
                vid[r] = -1; t_in[r] = INFINITY; t_out[r] = INFINITY;
                occlusion[r] = 0.0f;
                if (distance) { distance[r] = 0.0f; dist_total[r] = 0.0f; }
                if (normal) for (int a = 0; a < 3; ++a) { normal[3 * r + a] = 0.0f; albedo[3 * r + a] = 0.0f; }
                if (material) for (int a = 0; a < 4; ++a) material[4 * r + a] = 0.0f;
                if (raw_logits) for (int j = 0; j < NIFO_N_OUT; ++j) raw_logits[NIFO_N_OUT * r + j] = 0.0f;
                if (dist_accum) dist_accum[r] = 0.0f;
                st = 0;
                break;
            }
            /* evaluate the network on this voxel: reuse the single-voxel pipeline on a one-ray batch whose
               traversal result is forced to (id, ti, to) */
            nifo_eval_voxel(lattice, nv, theta_max, bend_k, nd, table, weights, o, d, flags, id, ti, to,
                            vid + r, t_in + r, t_out + r, occlusion + r, distance ? distance + r : 0,
                            dist_total ? dist_total + r : 0, normal ? normal + 3 * r : 0, albedo ? albedo + 3 * r : 0,
                            material ? material + 4 * r : 0, raw_logits ? raw_logits + NIFO_N_OUT * r : 0);
            ++k;
            float delta = ti - prev_exit, ell = to - ti;     /* unit direction: lengths = parameter differences */
            if (occlusion[r] >= 0.5f) {                      /* first voxel containing a hit: k */
                float tk = distance ? distance[r] : 0.0f;    /* t_k = sigmoid(z1) * (t_out - t_in) (R14) */
                if (dist_accum) dist_accum[r] = acc + delta + tk;
                st = 1;
                break;
            }
            acc += delta + ell;
            prev_exit = to;
            after_t = ti; after_id = id;
            if (k >= max_steps) { if (dist_accum) dist_accum[r] = acc; st = 2; break; }
        }
        status[r] = st; steps[r] = k;
    }
    return 0;
}

/* O11 trace: the first `max_steps` voxels of each ray's (t_in, id)-ordered sequence with the occlusion
   logit z0 the network predicts on each, WITHOUT stopping at an accepted voxel.  trace_id = -1 past
   the end of the sequence.  Tests use it to tell rays whose accept decisions are clear of the
   threshold (the CUDA path must agree exactly) from rays with a logit within rounding of 0 (where
   the fp16 path may legitimately decide the other way and any consistent outcome is valid). */
int nifo_walk_trace(int nv, const uint8_t* occ, const float* lattice, const void* bvh,
                    float theta_max, float bend_k,
                    const nifo_net_desc* nd, const float* table, const float* const* weights,
                    int64_t n, const float* origin, const float* dir, uint32_t flags, int max_steps,
                    int32_t* trace_id, float* trace_z0)
{
    for (int64_t r = 0; r < n; ++r) {
        const float* o = origin + 3 * r; const float* d = dir + 3 * r;
        float after_t = -INFINITY; int32_t after_id = -1;
        int k = 0;
        for (; k < max_steps; ++k) {
            int32_t id; float ti, to;
            if (bvh) traverse_bvh_after((const obvh*)bvh, o, d, after_t, after_id, &id, &ti, &to);
            else nifo_next_voxel_brute(nv, occ, lattice, 1, o, d, &after_t, &after_id, &id, &ti, &to);
            if (id < 0) break;
            int32_t v; float a, b, occl, raw[NIFO_N_OUT];
            nifo_eval_voxel(lattice, nv, theta_max, bend_k, nd, table, weights, o, d, NIFO_FLAG_OCCLUSION_ONLY | (flags & NIFO_FLAG_LATTICE_INVERSE), id, ti, to,
                            &v, &a, &b, &occl, 0, 0, 0, 0, 0, raw);
            trace_id[r * max_steps + k] = id; trace_z0[r * max_steps + k] = raw[0];
            after_t = ti; after_id = id;
        }
        for (; k < max_steps; ++k) { trace_id[r * max_steps + k] = -1; trace_z0[r * max_steps + k] = 0.0f; }
    }
    return 0;
}

/* O12  Hit positions ("During evaluation, we reconstruct hit positions along the same segmented
   ray in rest space").  From the outputs of the query: in deformed space the hit lies on the straight
   ray at the accumulated distance, x = o + D d (one fma per coordinate); in rest space it lies on the
   straight segment between the rest images of the voxel's entry and exit points (the local linear
   approximation of P:43) at the fraction u = clamp(distance / l, 0, 1) of the segment (u = 0 if l = 0).
   Miss: zeros (R18). */
void nifo_hit_positions(const float* lattice, int nv, uint32_t flags,
                        float theta_max, float bend_k, int64_t n, const float* origin, const float* dir,
                        const int32_t* vid, const float* t_in, const float* t_out,
                        const float* distance, const float* dist_total, float* hit_pos, float* hit_rest)
{
    for (int64_t r = 0; r < n; ++r) {
        const float* o = origin + 3 * r; const float* d = dir + 3 * r;
        if (vid[r] < 0) { for (int a = 0; a < 3; ++a) { hit_pos[3 * r + a] = 0.0f; hit_rest[3 * r + a] = 0.0f; } continue; }
        float Pi[3], Po[3], ri[3], ro[3];
        for (int a = 0; a < 3; ++a) {
            hit_pos[3 * r + a] = fmaf(dist_total[r], d[a], o[a]);
            Pi[a] = fmaf(t_in[r], d[a], o[a]); Po[a] = fmaf(t_out[r], d[a], o[a]);
        }
        if (flags & NIFO_FLAG_LATTICE_INVERSE) {
            inverse_trilinear_f32(lattice, nv, vid[r], Pi, ri);
            inverse_trilinear_f32(lattice, nv, vid[r], Po, ro);
        } else {
            inverse_f32(theta_max, bend_k, Pi, ri);
            inverse_f32(theta_max, bend_k, Po, ro);
        }
        float ell = t_out[r] - t_in[r];
        float u = ell > 0.0f ? distance[r] / ell : 0.0f;
        u = u < 0.0f ? 0.0f : (u > 1.0f ? 1.0f : u);
        for (int a = 0; a < 3; ++a) hit_rest[3 * r + a] = fmaf(u, ro[a] - ri[a], ri[a]);
    }
}

/* rest-space normalised endpoints of hit rays (exposed for the "inside the hit voxel's rest
   cell" invariant): out[r*6 + e*3 + a]; NaN for a miss. */
void nifo_rest_endpoints(float theta_max, float bend_k, int64_t n, const float* origin,
                         const float* dir, const int32_t* vid, const float* t_in,
                         const float* t_out, float* out)
{
    for (int64_t r = 0; r < n; ++r)
        for (int e = 0; e < 2; ++e) {
            float P[3], pr[3];
            float t = e ? t_out[r] : t_in[r];
            for (int a = 0; a < 3; ++a) P[a] = fmaf(t, dir[3 * r + a], origin[3 * r + a]);
            if (vid[r] < 0) { pr[0] = pr[1] = pr[2] = NAN; }
            else inverse_f32(theta_max, bend_k, P, pr);
            for (int a = 0; a < 3; ++a) out[6 * r + 3 * e + a] = pr[a];
        }
}
