/*
 * pn_gen_oracle.c -- CPU oracle of the on-device initial-data generator.
 * TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build or call it.  It shares no code with the CUDA path.
 *
 * What it computes (plain C, double, one loop over systems, libm sin/cos/sqrt):
 *   the paper draws, for every inspiral, random initial spin orientations uniform on the sphere with
 *   L^ = (0,0,1) and M = 1 ("generated on the GPU").  The recipe is the
 *   one of DESIGN.md 5 (the same as paper_0908_3889_b200/workloads.py, which draws it with numpy's own
 *   Philox generator): seven uniform variates per system, in the order q, chi1, chi2, z1, phi1, z2, phi2,
 *   each variate column k being the k-th length-N_total block of ONE counter-based stream:
 *       variate (k, i) = U(raw[k*N_total + i]),  U(x) = (x >> 11) * 2^-53,
 *       raw[e] = word (e mod 4) of Philox4x64-10(counter = e/4 + 1, key)          (numpy's Philox layout)
 *   q = q_lo + (q_hi-q_lo) u (q_lo if q_hi <= q_lo), chi_i likewise; unit vectors from z = 2u-1,
 *   phi = 2 pi u', (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z) -- exactly uniform on the sphere, the same
 *   distribution as the paper's Marsaglia sampler [21] (R17); m1 = 1/(1+q), m2 = q/(1+q) or
 *   (m1_fixed, 1 - m1_fixed); S_i = ((chi_i m_i) m_i) S^_i; optionally S^_1 fixed at
 *   (sin t, 0, cos t).  State layout y = (omega0, S1, S2, 0, 0, 1).
 *
 * Philox4x64-10 is the counter-based generator of Salmon et al. (SC'11) as used by numpy.random.Philox:
 * ten rounds of two 64x64->128 multiplications with the key bumped by Weyl constants between rounds,
 * written out below from its definition.
 *
 * Pins (tests/test_oracle_gen.py): raw words against numpy.random.Philox(key=..., counter=...).random_raw
 * (an independent implementation), variates against numpy.random.Generator.random, full states against
 * workloads.generate for all five configs, uniformity / isotropy moments.  Parity unpinned: none.
 */
#include <math.h>
#include <stdint.h>

typedef unsigned __int128 u128;

#define PHILOX_M0 0xD2E7470EE14C6C93ULL
#define PHILOX_M1 0xCA5A826395121157ULL
#define PHILOX_W0 0x9E3779B97F4A7C15ULL /* golden ratio */
#define PHILOX_W1 0xBB67AE8584CAA73BULL /* sqrt(3) - 1 */

/* one Philox4x64 evaluation, 10 rounds; ctr and key are not modified */
void pn_gen_oracle_philox4x64_10(const uint64_t ctr[4], const uint64_t key[2], uint64_t out[4])
{
    uint64_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint64_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += PHILOX_W0; k1 += PHILOX_W1; }
        const u128 p0 = (u128)PHILOX_M0 * c0;
        const u128 p1 = (u128)PHILOX_M1 * c2;
        const uint64_t hi0 = (uint64_t)(p0 >> 64), lo0 = (uint64_t)p0;
        const uint64_t hi1 = (uint64_t)(p1 >> 64), lo1 = (uint64_t)p1;
        const uint64_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* raw[e] of the stream (numpy layout: the counter is incremented BEFORE each block of four words) */
uint64_t pn_gen_oracle_raw(const uint64_t key[2], uint64_t e)
{
    const uint64_t ctr[4] = {e / 4 + 1, 0, 0, 0};
    uint64_t out[4];
    pn_gen_oracle_philox4x64_10(ctr, key, out);
    return out[e % 4];
}

double pn_gen_oracle_uniform(const uint64_t key[2], uint64_t e)
{
    return (double)(pn_gen_oracle_raw(key, e) >> 11) * (1.0 / 9007199254740992.0);
}

void pn_gen_oracle_raw_block(const uint64_t key[2], uint64_t first, long long n, uint64_t *out)
{
    for (long long j = 0; j < n; ++j) out[j] = pn_gen_oracle_raw(key, first + (uint64_t)j);
}

typedef struct {
    uint64_t key[2];
    double omega0;
    double q_lo, q_hi;
    double m1_fixed;            /* > 0: m1 = m1_fixed, m2 = 1 - m1_fixed */
    double chi1_lo, chi1_hi, chi2_lo, chi2_hi;
    double s1_tilt_deg;         /* >= 0: S^_1 = (sin t, 0, cos t); < 0: isotropic */
} pn_gen_spec;

static double lerp_or_fixed(double lo, double hi, double u) { return hi > lo ? lo + (hi - lo) * u : lo; }

/* systems first .. first+count-1 of an ensemble of n_total systems */
void pn_gen_oracle_generate(const pn_gen_spec *s, long long n_total, long long first, long long count,
                            double *init_states /*[count][10]*/, double *masses /*[count][2]*/)
{
    const double two_pi = 2.0 * 3.14159265358979323846;
    for (long long j = 0; j < count; ++j) {
        const uint64_t i = (uint64_t)(first + j), N = (uint64_t)n_total;
        double u[7];
        for (int k = 0; k < 7; ++k) u[k] = pn_gen_oracle_uniform(s->key, (uint64_t)k * N + i);
        const double q = lerp_or_fixed(s->q_lo, s->q_hi, u[0]);
        const double chi1 = lerp_or_fixed(s->chi1_lo, s->chi1_hi, u[1]);
        const double chi2 = lerp_or_fixed(s->chi2_lo, s->chi2_hi, u[2]);
        double s1[3], s2[3];
        {
            const double z = 2.0 * u[3] - 1.0, phi = two_pi * u[4];
            const double r = sqrt(fmax(0.0, 1.0 - z * z));
            s1[0] = r * cos(phi); s1[1] = r * sin(phi); s1[2] = z;
        }
        {
            const double z = 2.0 * u[5] - 1.0, phi = two_pi * u[6];
            const double r = sqrt(fmax(0.0, 1.0 - z * z));
            s2[0] = r * cos(phi); s2[1] = r * sin(phi); s2[2] = z;
        }
        double m1, m2;
        if (s->m1_fixed > 0.0) { m1 = s->m1_fixed; m2 = 1.0 - m1; }
        else { m1 = 1.0 / (1.0 + q); m2 = q / (1.0 + q); }
        if (s->s1_tilt_deg >= 0.0) {
            const double th = s->s1_tilt_deg * (3.14159265358979323846 / 180.0);
            s1[0] = sin(th); s1[1] = 0.0; s1[2] = cos(th);
        }
        double *y = init_states + 10 * j;
        const double a1 = (chi1 * m1) * m1, a2 = (chi2 * m2) * m2;
        y[0] = s->omega0;
        for (int c = 0; c < 3; ++c) { y[1 + c] = a1 * s1[c]; y[4 + c] = a2 * s2[c]; }
        y[7] = 0.0; y[8] = 0.0; y[9] = 1.0;
        masses[2 * j] = m1; masses[2 * j + 1] = m2;
    }
}
