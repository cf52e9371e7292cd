/*
 * fenc_oracle.c -- CPU ORACLE for the FEnc^2 CKKS hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this file.  It shares no code, header, table or constant generator with the
 * CUDA library under paper_2606_16359_b200/csrc/, and never includes a CUDA header.
 *
 * Plain, slow, single-threaded C.  Every polynomial lives in the COEFFICIENT domain with
 * canonical residues in [0,q); a product of two polynomials is the negacyclic product in
 * Z_q[X]/(X^N+1) ("a degree-N polynomial in Z_q[X]/(X^N+1)").  The paper only
 * names the CKKS primitives (Eq. 1); their RNS form follows the readings of
 * DESIGN.md section 4, cited per function as "R2.x".
 *
 * Pins (tests/test_oracle_*.py): NTT product vs schoolbook negacyclic product; ModUp/ModDown/
 * rescale vs exact big-integer characterisations in Python; rotation = cyclic slot shift.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef uint64_t u64;
typedef unsigned __int128 u128;

#define ORC_MAXLIMB 96 /* config 5's largest point: 36 ciphertext + 36 special limbs */

/* ------------------------------------------------------------------ modular scalars */
u64 orc_mulmod(u64 a, u64 b, u64 q) { return (u64)(((u128)a * b) % q); }
u64 orc_addmod(u64 a, u64 b, u64 q) { u64 s = a + b; return (s >= q) ? s - q : s; } /* q < 2^63 */
u64 orc_submod(u64 a, u64 b, u64 q) { return (a >= b) ? a - b : a + q - b; }
u64 orc_powmod(u64 a, u64 e, u64 q) {
    u64 r = 1 % q; a %= q;
    while (e) { if (e & 1) r = orc_mulmod(r, a, q); a = orc_mulmod(a, a, q); e >>= 1; }
    return r;
}
u64 orc_invmod(u64 a, u64 q) { return orc_powmod(a, q - 2, q); } /* q prime */

/* ------------------------------------------------------------------ NTT (R2.1)
 * NTT(a)[e] = sum_i a_i psi^{(2e+1) i} mod q, e in [0,N), natural order.
 * Computed as: b_i = a_i psi^i, then the cyclic DFT of b with omega = psi^2 by the
 * textbook iterative radix-2 algorithm (bit-reversal copy, then log2 N butterfly levels,
 * twiddles by repeated multiplication).  No tables. */
static unsigned bitrev(unsigned x, int bits) {
    unsigned r = 0; for (int i = 0; i < bits; i++) { r = (r << 1) | (x & 1); x >>= 1; } return r;
}
static void cyclic_dft(size_t N, u64 q, u64 omega, u64 *a) {
    int bits = 0; while (((size_t)1 << bits) < N) bits++;
    for (size_t i = 0; i < N; i++) { size_t j = bitrev((unsigned)i, bits); if (i < j) { u64 t = a[i]; a[i] = a[j]; a[j] = t; } }
    for (size_t len = 2; len <= N; len <<= 1) {
        u64 wlen = orc_powmod(omega, N / len, q);
        for (size_t s = 0; s < N; s += len) {
            u64 w = 1;
            for (size_t k = 0; k < len / 2; k++) {
                u64 x = a[s + k], y = orc_mulmod(a[s + k + len / 2], w, q);
                a[s + k] = orc_addmod(x, y, q);
                a[s + k + len / 2] = orc_submod(x, y, q);
                w = orc_mulmod(w, wlen, q);
            }
        }
    }
}
void orc_ntt(size_t N, u64 q, u64 psi, u64 *a) {
    u64 w = 1;
    for (size_t i = 0; i < N; i++) { a[i] = orc_mulmod(a[i], w, q); w = orc_mulmod(w, psi, q); }
    cyclic_dft(N, q, orc_mulmod(psi, psi, q), a);
}
void orc_intt(size_t N, u64 q, u64 psi, u64 *a) {
    u64 ipsi = orc_invmod(psi, q), ninv = orc_invmod((u64)N % q, q);
    cyclic_dft(N, q, orc_mulmod(ipsi, ipsi, q), a);
    u64 w = ninv;
    for (size_t i = 0; i < N; i++) { a[i] = orc_mulmod(a[i], w, q); w = orc_mulmod(w, ipsi, q); }
}

/* negacyclic product c = a * b in Z_q[X]/(X^N+1) through the NTT (R2.1) */
void orc_polymul(size_t N, u64 q, u64 psi, const u64 *a, const u64 *b, u64 *c) {
    u64 *x = malloc(N * sizeof(u64)), *y = malloc(N * sizeof(u64));
    memcpy(x, a, N * sizeof(u64)); memcpy(y, b, N * sizeof(u64));
    orc_ntt(N, q, psi, x); orc_ntt(N, q, psi, y);
    for (size_t i = 0; i < N; i++) x[i] = orc_mulmod(x[i], y[i], q);
    orc_intt(N, q, psi, x);
    memcpy(c, x, N * sizeof(u64));
    free(x); free(y);
}
/* the slow definition: c_k = sum_{i+j=k} a_i b_j - sum_{i+j=k+N} a_i b_j  (R2.1) */
void orc_schoolbook(size_t N, u64 q, const u64 *a, const u64 *b, u64 *c) {
    for (size_t k = 0; k < N; k++) c[k] = 0;
    for (size_t i = 0; i < N; i++) for (size_t j = 0; j < N; j++) {
        u64 p = orc_mulmod(a[i], b[j], q); size_t k = i + j;
        if (k < N) c[k] = orc_addmod(c[k], p, q); else c[k - N] = orc_submod(c[k - N], p, q);
    }
}

/* ------------------------------------------------------------------ automorphism (R2.7)
 * sigma_g: a(X) -> a(X^g): coefficient i moves to index i*g mod 2N; an index >= N lands
 * at index-N negated. */
void orc_automorph(size_t N, u64 q, u64 g, const u64 *in, u64 *out) {
    for (size_t i = 0; i < N; i++) {
        size_t k = (size_t)(((u128)i * g) % (2 * N));
        if (k < N) out[k] = in[i]; else out[k - N] = in[i] ? q - in[i] : 0;
    }
}

/* ------------------------------------------------------------------ parameter block */
typedef struct {
    size_t N; int nq, np, dlen;
    u64 mod[ORC_MAXLIMB];  /* q_0..q_{nq-1}, then p_0..p_{np-1} */
    u64 psi[ORC_MAXLIMB];  /* a primitive 2N-th root of unity per modulus */
} orc_params;

orc_params *orc_params_new(size_t N, int nq, const u64 *q, const u64 *psi_q, int np, const u64 *p, const u64 *psi_p, int dlen) {
    if (nq + np > ORC_MAXLIMB) return NULL;
    orc_params *P = calloc(1, sizeof *P);
    P->N = N; P->nq = nq; P->np = np; P->dlen = dlen;
    for (int i = 0; i < nq; i++) { P->mod[i] = q[i]; P->psi[i] = psi_q[i]; }
    for (int i = 0; i < np; i++) { P->mod[nq + i] = p[i]; P->psi[nq + i] = psi_p[i]; }
    return P;
}
void orc_params_free(orc_params *P) { free(P); }

/* Extended-basis arrays used below have "E = L + np" rows: rows 0..L-1 are q_0..q_{L-1},
 * rows L..L+np-1 are p_0..p_{np-1}.  ext_mod maps such a row to its index in P->mod. */
static int ext_mod(const orc_params *P, int L, int row) { return row < L ? row : P->nq + (row - L); }

/* ------------------------------------------------------------------ ModUp (R2.6)
 * digit j = limbs [j*dlen, min((j+1)*dlen, L)); Q_j = product of the digit's primes.
 * target t in the digit: up[t] = d[t];  otherwise
 *   y_i = d[q_i] * [(Q_j/q_i)^{-1}]_{q_i} mod q_i,  up[t] = ( sum_i y_i * ((Q_j/q_i) mod t) ) mod t.
 * No floating-point or centring correction.  d: [L][N]; up: [L+np][N]. */
void orc_modup(const orc_params *P, int L, int j, const u64 *d, u64 *up) {
    size_t N = P->N; int lo = j * P->dlen, hi = lo + P->dlen; if (hi > L) hi = L;
    int E = L + P->np;
    u64 *y = malloc((size_t)(hi - lo) * N * sizeof(u64));
    for (int i = lo; i < hi; i++) {
        u64 qi = P->mod[i], qhat = 1;
        for (int i2 = lo; i2 < hi; i2++) if (i2 != i) qhat = orc_mulmod(qhat, P->mod[i2] % qi, qi);
        u64 inv = orc_invmod(qhat, qi);
        for (size_t n = 0; n < N; n++) y[(size_t)(i - lo) * N + n] = orc_mulmod(d[(size_t)i * N + n], inv, qi);
    }
    for (int row = 0; row < E; row++) {
        u64 *dst = up + (size_t)row * N;
        if (row >= lo && row < hi) { memcpy(dst, d + (size_t)row * N, N * sizeof(u64)); continue; }
        u64 t = P->mod[ext_mod(P, L, row)];
        for (size_t n = 0; n < N; n++) dst[n] = 0;
        for (int i = lo; i < hi; i++) {
            u64 qhat_t = 1;
            for (int i2 = lo; i2 < hi; i2++) if (i2 != i) qhat_t = orc_mulmod(qhat_t, P->mod[i2] % t, t);
            for (size_t n = 0; n < N; n++)
                dst[n] = orc_addmod(dst[n], orc_mulmod(y[(size_t)(i - lo) * N + n] % t, qhat_t, t), t);
        }
    }
    free(y);
}

/* ------------------------------------------------------------------ ModDown (R2.6)
 * y_i = acc[p_i] * [(P/p_i)^{-1}]_{p_i};  conv[t] = ( sum_i y_i * ((P/p_i) mod t) ) mod t;
 * out[t] = (acc[t] - conv[t]) * [P^{-1}]_t mod t, t in q_0..q_{L-1}.  acc: [L+np][N]; out: [L][N]. */
void orc_moddown(const orc_params *P, int L, const u64 *acc, u64 *out) {
    size_t N = P->N; int np = P->np;
    u64 *y = malloc((size_t)np * N * sizeof(u64));
    for (int i = 0; i < np; i++) {
        u64 pi = P->mod[P->nq + i], phat = 1;
        for (int i2 = 0; i2 < np; i2++) if (i2 != i) phat = orc_mulmod(phat, P->mod[P->nq + i2] % pi, pi);
        u64 inv = orc_invmod(phat, pi);
        for (size_t n = 0; n < N; n++) y[(size_t)i * N + n] = orc_mulmod(acc[(size_t)(L + i) * N + n], inv, pi);
    }
    for (int t = 0; t < L; t++) {
        u64 q = P->mod[t], Pmod = 1;
        for (int i = 0; i < np; i++) Pmod = orc_mulmod(Pmod, P->mod[P->nq + i] % q, q);
        u64 Pinv = orc_invmod(Pmod, q);
        for (size_t n = 0; n < N; n++) {
            u64 conv = 0;
            for (int i = 0; i < np; i++) {
                u64 phat_t = 1;
                for (int i2 = 0; i2 < np; i2++) if (i2 != i) phat_t = orc_mulmod(phat_t, P->mod[P->nq + i2] % q, q);
                conv = orc_addmod(conv, orc_mulmod(y[(size_t)i * N + n] % q, phat_t, q), q);
            }
            out[(size_t)t * N + n] = orc_mulmod(orc_submod(acc[(size_t)t * N + n], conv, q), Pinv, q);
        }
    }
    free(y);
}

/* ------------------------------------------------------------------ hybrid key switch (R2.6)
 * d: [L][N].  key_b, key_a: [beta_max][nq+np][N] over ALL limbs (level independent);
 * beta = ceil(L/dlen) digits are used.  acc_0[t] = sum_j up_j[t] * b_j[t], acc_1 likewise,
 * over the L+np limbs in use, then ModDown of each.  out0, out1: [L][N]. */
void orc_keyswitch(const orc_params *P, int L, const u64 *d, const u64 *key_b, const u64 *key_a, u64 *out0, u64 *out1) {
    size_t N = P->N; int E = L + P->np, A = P->nq + P->np;
    int beta = (L + P->dlen - 1) / P->dlen;
    u64 *up = malloc((size_t)E * N * sizeof(u64));
    u64 *acc0 = calloc((size_t)E * N, sizeof(u64)), *acc1 = calloc((size_t)E * N, sizeof(u64));
    u64 *prod = malloc(N * sizeof(u64));
    for (int j = 0; j < beta; j++) {
        orc_modup(P, L, j, d, up);
        for (int row = 0; row < E; row++) {
            int mi = ext_mod(P, L, row); u64 t = P->mod[mi], psi = P->psi[mi];
            const u64 *kb = key_b + ((size_t)j * A + mi) * N, *ka = key_a + ((size_t)j * A + mi) * N;
            orc_polymul(N, t, psi, up + (size_t)row * N, kb, prod);
            for (size_t n = 0; n < N; n++) acc0[(size_t)row * N + n] = orc_addmod(acc0[(size_t)row * N + n], prod[n], t);
            orc_polymul(N, t, psi, up + (size_t)row * N, ka, prod);
            for (size_t n = 0; n < N; n++) acc1[(size_t)row * N + n] = orc_addmod(acc1[(size_t)row * N + n], prod[n], t);
        }
    }
    orc_moddown(P, L, acc0, out0);
    orc_moddown(P, L, acc1, out1);
    free(up); free(acc0); free(acc1); free(prod);
}

/* ------------------------------------------------------------------ rotation (R2.7, Eq. 1)
 * Rot(ct, r): g = 5^r mod 2N (passed in).  sigma_g on c0 and c1 FIRST, then
 * (ks0, ks1) = KS(sigma_g(c1); rotkey), result (sigma_g(c0) + ks0, ks1).  ct: [2][L][N]. */
void orc_rotate(const orc_params *P, int L, u64 g, const u64 *ct, const u64 *key_b, const u64 *key_a, u64 *out) {
    size_t N = P->N, LN = (size_t)L * N;
    u64 *s0 = malloc(LN * sizeof(u64)), *s1 = malloc(LN * sizeof(u64));
    for (int t = 0; t < L; t++) {
        orc_automorph(N, P->mod[t], g, ct + (size_t)t * N, s0 + (size_t)t * N);
        orc_automorph(N, P->mod[t], g, ct + LN + (size_t)t * N, s1 + (size_t)t * N);
    }
    orc_keyswitch(P, L, s1, key_b, key_a, out, out + LN);
    for (int t = 0; t < L; t++) for (size_t n = 0; n < N; n++)
        out[(size_t)t * N + n] = orc_addmod(out[(size_t)t * N + n], s0[(size_t)t * N + n], P->mod[t]);
    free(s0); free(s1);
}

/* ------------------------------------------------------------------ hoisted rotation (R2.7b)
 * Several rotations of ONE ciphertext share the decomposition: up_j = ModUp_j(c1) is computed from the UNROTATED c1,
 * and each rotation applies sigma_g to the extended digits instead of to c1:
 *   acc_0[t] = sum_j sigma_g(up_j)[t] * b_j[t], acc_1 likewise;  result (sigma_g(c0) + ModDown(acc_0), ModDown(acc_1)).
 * sigma_g(up_j) is congruent to sigma_g(c1) modulo the digit's primes and differs from ModUp_j(sigma_g(c1)) by a
 * small multiple of Q_j on the other limbs, so the result decrypts to the same rotation with key-switch noise of the
 * same size, but its limbs are NOT those of orc_rotate.  Same keys as orc_rotate. */
void orc_rotate_hoisted(const orc_params *P, int L, u64 g, const u64 *ct, const u64 *key_b, const u64 *key_a, u64 *out) {
    size_t N = P->N, LN = (size_t)L * N; int E = L + P->np, A = P->nq + P->np;
    int beta = (L + P->dlen - 1) / P->dlen;
    u64 *up = malloc((size_t)E * N * sizeof(u64)), *rot = malloc(N * sizeof(u64)), *prod = malloc(N * sizeof(u64));
    u64 *acc0 = calloc((size_t)E * N, sizeof(u64)), *acc1 = calloc((size_t)E * N, sizeof(u64));
    for (int j = 0; j < beta; j++) {
        orc_modup(P, L, j, ct + LN, up);
        for (int row = 0; row < E; row++) {
            int mi = ext_mod(P, L, row); u64 t = P->mod[mi], psi = P->psi[mi];
            const u64 *kb = key_b + ((size_t)j * A + mi) * N, *ka = key_a + ((size_t)j * A + mi) * N;
            orc_automorph(N, t, g, up + (size_t)row * N, rot);
            orc_polymul(N, t, psi, rot, kb, prod);
            for (size_t n = 0; n < N; n++) acc0[(size_t)row * N + n] = orc_addmod(acc0[(size_t)row * N + n], prod[n], t);
            orc_polymul(N, t, psi, rot, ka, prod);
            for (size_t n = 0; n < N; n++) acc1[(size_t)row * N + n] = orc_addmod(acc1[(size_t)row * N + n], prod[n], t);
        }
    }
    orc_moddown(P, L, acc0, out);
    orc_moddown(P, L, acc1, out + LN);
    for (int t = 0; t < L; t++) {
        orc_automorph(N, P->mod[t], g, ct + (size_t)t * N, rot);
        for (size_t n = 0; n < N; n++) out[(size_t)t * N + n] = orc_addmod(out[(size_t)t * N + n], rot[n], P->mod[t]);
    }
    free(up); free(rot); free(prod); free(acc0); free(acc1);
}

/* ------------------------------------------------------------------ Add / PMult / Rescale (R2.8) */
void orc_add(const orc_params *P, int L, int npoly, const u64 *a, const u64 *b, u64 *out) {
    size_t N = P->N;
    for (int k = 0; k < npoly; k++) for (int t = 0; t < L; t++) for (size_t n = 0; n < N; n++) {
        size_t o = ((size_t)k * L + t) * N + n; out[o] = orc_addmod(a[o], b[o], P->mod[t]);
    }
}
/* acc += ct (*) pt on both polynomials, limb by limb; ct, acc: [2][L][N], pt: [L][N] */
void orc_pmult_acc(const orc_params *P, int L, const u64 *ct, const u64 *pt, u64 *acc) {
    size_t N = P->N; u64 *prod = malloc(N * sizeof(u64));
    for (int k = 0; k < 2; k++) for (int t = 0; t < L; t++) {
        size_t o = ((size_t)k * L + t) * N;
        orc_polymul(N, P->mod[t], P->psi[t], ct + o, pt + (size_t)t * N, prod);
        for (size_t n = 0; n < N; n++) acc[o + n] = orc_addmod(acc[o + n], prod[n], P->mod[t]);
    }
    free(prod);
}
/* one polynomial product per limb: out[t] = a[t] * b[t]; a, b, out: [L][N] */
void orc_polymul_rns(const orc_params *P, int L, const u64 *a, const u64 *b, u64 *out) {
    for (int t = 0; t < L; t++)
        orc_polymul(P->N, P->mod[t], P->psi[t], a + (size_t)t * P->N, b + (size_t)t * P->N, out + (size_t)t * P->N);
}
/* Rescale: drop limb q_{L-1}: c'[t] = (c[t] - (c[q_{L-1}] mod t)) * [q_{L-1}^{-1}]_t mod t, i.e. exact
 * floor(C / q_{L-1}) on the canonical non-negative representative (reading A10).  c: [L][N] -> out: [L-1][N]. */
void orc_rescale(const orc_params *P, int L, const u64 *c, u64 *out) {
    size_t N = P->N; u64 ql = P->mod[L - 1];
    for (int t = 0; t < L - 1; t++) {
        u64 q = P->mod[t], inv = orc_invmod(ql % q, q);
        for (size_t n = 0; n < N; n++)
            out[(size_t)t * N + n] = orc_mulmod(orc_submod(c[(size_t)t * N + n], c[(size_t)(L - 1) * N + n] % q, q), inv, q);
    }
}
/* every limb of a polynomial times the integer scalar k (given reduced per limb: k_t = k mod q_t) */
void orc_mul_scalar(const orc_params *P, int L, const u64 *a, const u64 *k_t, u64 *out) {
    for (int t = 0; t < L; t++) for (size_t n = 0; n < P->N; n++)
        out[(size_t)t * P->N + n] = orc_mulmod(a[(size_t)t * P->N + n], k_t[t], P->mod[t]);
}
/* reduce centred signed integer coefficients into L limbs (negative -> q - |m|) (R2.2) */
void orc_reduce_signed(const orc_params *P, int L, const int64_t *m, u64 *out) {
    for (int t = 0; t < L; t++) { u64 q = P->mod[t];
        for (size_t n = 0; n < P->N; n++) { int64_t v = m[n];
            out[(size_t)t * P->N + n] = v >= 0 ? (u64)v % q : (q - ((u64)(-v) % q)) % q; } }
}
