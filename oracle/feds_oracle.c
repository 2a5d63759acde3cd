/*
 * feds_oracle.c — plain, slow, obviously-correct CPU ORACLE for the selective-encryption
 * fragmentation path of arXiv 1512.02951 §6 (PAPER.md; "P:n" = PAPER.md line n).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT. Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference arm may build, load or call it. It shares no code, table or
 * constant generator with the CUDA path (paper_1512_02951_b200/csrc); neither includes the other.
 *
 * Every step is the textbook definition written out, in double precision / exact integers, in the
 * paper's order; there is no blocking, fusion, table-driven shortcut or reordering:
 *   - DCT/IDCT 8x8: the defining double sum (scaling pinned by P:568 "DC <= 2040").
 *   - zigzag select: anti-diagonal walk reproducing P:494's default selection.
 *   - AES-128: FIPS-197 as written (S-box from GF(2^8) inverse + affine map, ShiftRows, MixColumns
 *     with xtime, key expansion with Rcon); CTR per SP 800-38A 6.5 with a 128-bit big-endian
 *     increment ("AES 128-bit", "counter mode"; counter format = DESIGN.md A6).
 *   - SHA-256: FIPS 180-4 6.2 as written; Merkle layout = DESIGN.md 2.1 / 2.2 (A9).
 *   - 5/3 DWT: integer lifting P:755-762 eq. (1)-(2) in the DESIGN.md A12 reading, rows then
 *     columns, level shift -128, whole-sample symmetric extension (A14).
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py (standards' known-answer
 * vectors, closed forms, hashlib / cryptography / scipy cross-checks, brute force). Parity with the
 * paper authors' own (unavailable) code is unpinned and not needed.
 *
 * All functions are extern "C"-style plain C; all pointers are HOST pointers; nothing is allocated
 * that is not freed before return; return value 0 = ok, negative = argument error.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------ */
/* SHA-256 — FIPS 180-4 section 6.2                                                             */
/* ------------------------------------------------------------------------------------------ */

static uint32_t rotr32(uint32_t x, int n) { return (x >> n) | (x << (32 - n)); }

/* FIPS 180-4 4.2.2: first 32 bits of the fractional parts of the cube roots of the first 64 primes */
static const uint32_t SHA256_K[64] = {
    0x428a2f98, 0x71374491, 0xb5c0fbcf, 0xe9b5dba5, 0x3956c25b, 0x59f111f1, 0x923f82a4, 0xab1c5ed5,
    0xd807aa98, 0x12835b01, 0x243185be, 0x550c7dc3, 0x72be5d74, 0x80deb1fe, 0x9bdc06a7, 0xc19bf174,
    0xe49b69c1, 0xefbe4786, 0x0fc19dc6, 0x240ca1cc, 0x2de92c6f, 0x4a7484aa, 0x5cb0a9dc, 0x76f988da,
    0x983e5152, 0xa831c66d, 0xb00327c8, 0xbf597fc7, 0xc6e00bf3, 0xd5a79147, 0x06ca6351, 0x14292967,
    0x27b70a85, 0x2e1b2138, 0x4d2c6dfc, 0x53380d13, 0x650a7354, 0x766a0abb, 0x81c2c92e, 0x92722c85,
    0xa2bfe8a1, 0xa81a664b, 0xc24b8b70, 0xc76c51a3, 0xd192e819, 0xd6990624, 0xf40e3585, 0x106aa070,
    0x19a4c116, 0x1e376c08, 0x2748774c, 0x34b0bcb5, 0x391c0cb3, 0x4ed8aa4a, 0x5b9cca4f, 0x682e6ff3,
    0x748f82ee, 0x78a5636f, 0x84c87814, 0x8cc70208, 0x90befffa, 0xa4506ceb, 0xbef9a3f7, 0xc67178f2};

/* one 512-bit block, FIPS 180-4 6.2.2 steps 1-4 */
static void sha256_block(uint32_t H[8], const uint8_t M[64]) {
    uint32_t W[64];
    for (int t = 0; t < 16; t++)
        W[t] = ((uint32_t)M[4 * t] << 24) | ((uint32_t)M[4 * t + 1] << 16) | ((uint32_t)M[4 * t + 2] << 8) |
               (uint32_t)M[4 * t + 3];
    for (int t = 16; t < 64; t++) {
        uint32_t s0 = rotr32(W[t - 15], 7) ^ rotr32(W[t - 15], 18) ^ (W[t - 15] >> 3);
        uint32_t s1 = rotr32(W[t - 2], 17) ^ rotr32(W[t - 2], 19) ^ (W[t - 2] >> 10);
        W[t] = s1 + W[t - 7] + s0 + W[t - 16];
    }
    uint32_t a = H[0], b = H[1], c = H[2], d = H[3], e = H[4], f = H[5], g = H[6], h = H[7];
    for (int t = 0; t < 64; t++) {
        uint32_t S1 = rotr32(e, 6) ^ rotr32(e, 11) ^ rotr32(e, 25);
        uint32_t ch = (e & f) ^ (~e & g);
        uint32_t T1 = h + S1 + ch + SHA256_K[t] + W[t];
        uint32_t S0 = rotr32(a, 2) ^ rotr32(a, 13) ^ rotr32(a, 22);
        uint32_t maj = (a & b) ^ (a & c) ^ (b & c);
        uint32_t T2 = S0 + maj;
        h = g; g = f; f = e; e = d + T1; d = c; c = b; b = a; a = T1 + T2;
    }
    H[0] += a; H[1] += b; H[2] += c; H[3] += d; H[4] += e; H[5] += f; H[6] += g; H[7] += h;
}

/* whole-message SHA-256: padding per FIPS 180-4 5.1.1, initial value 5.3.3 */
void orc_sha256(const uint8_t *msg, uint64_t n, uint8_t out[32]) {
    uint32_t H[8] = {0x6a09e667, 0xbb67ae85, 0x3c6ef372, 0xa54ff53a, 0x510e527f, 0x9b05688c, 0x1f83d9ab, 0x5be0cd19};
    uint64_t full = n / 64;
    for (uint64_t i = 0; i < full; i++) sha256_block(H, msg + 64 * i);
    uint8_t tail[128];
    uint64_t rem = n - 64 * full;
    memset(tail, 0, sizeof tail);
    if (rem) memcpy(tail, msg + 64 * full, rem);
    tail[rem] = 0x80;
    int tail_blocks = (rem + 1 + 8 <= 64) ? 1 : 2;
    uint64_t bits = n * 8;
    for (int i = 0; i < 8; i++) tail[64 * tail_blocks - 1 - i] = (uint8_t)(bits >> (8 * i));
    for (int i = 0; i < tail_blocks; i++) sha256_block(H, tail + 64 * i);
    for (int i = 0; i < 8; i++) {
        out[4 * i] = (uint8_t)(H[i] >> 24); out[4 * i + 1] = (uint8_t)(H[i] >> 16);
        out[4 * i + 2] = (uint8_t)(H[i] >> 8); out[4 * i + 3] = (uint8_t)H[i];
    }
}

/* Upper Merkle levels: n digests (32 B each, concatenated in `d`) -> root.
 * n == 0 -> SHA-256(""); n == 1 -> the digest itself; else nodes of <= F children, repeated. */
int orc_merkle_root(const uint8_t *d, uint64_t n, int F, uint8_t root[32]) {
    if (F < 2) return -1;
    if (n == 0) { orc_sha256((const uint8_t *)"", 0, root); return 0; }
    uint8_t *cur = (uint8_t *)malloc(32 * n);
    if (!cur) return -2;
    memcpy(cur, d, 32 * n);
    while (n > 1) {
        uint64_t m = (n + F - 1) / F;
        uint8_t *nxt = (uint8_t *)malloc(32 * m);
        for (uint64_t j = 0; j < m; j++) {
            uint64_t lo = j * F, hi = lo + F < n ? lo + F : n;
            orc_sha256(cur + 32 * lo, 32 * (hi - lo), nxt + 32 * j);
        }
        free(cur); cur = nxt; n = m;
    }
    memcpy(root, cur, 32);
    free(cur);
    return 0;
}

/* DWT-path digest: leaves are LEAF-byte runs of the stream. */
int orc_merkle_stream(const uint8_t *bytes, uint64_t n, uint64_t leaf_bytes, int F, uint8_t root[32]) {
    if (leaf_bytes == 0) return -1;
    uint64_t nl = (n + leaf_bytes - 1) / leaf_bytes;
    uint8_t *leaves = (uint8_t *)malloc(nl ? 32 * nl : 1);
    for (uint64_t j = 0; j < nl; j++) {
        uint64_t lo = j * leaf_bytes, hi = lo + leaf_bytes < n ? lo + leaf_bytes : n;
        orc_sha256(bytes + lo, hi - lo, leaves + 32 * j);
    }
    int rc = orc_merkle_root(leaves, nl, F, root);
    free(leaves);
    return rc;
}

/* DCT-path digest: a fragment holds `per_block` bytes for each of
 * n_rows = C*nbr block rows x nbc blocks; leaf (row, g) = bytes of blocks [g*G, min((g+1)*G, nbc)). */
int orc_merkle_blocks(const uint8_t *bytes, uint64_t n_rows, uint64_t nbc, uint64_t per_block, int G, int F,
                      uint8_t root[32]) {
    if (G < 1) return -1;
    if (per_block == 0 || n_rows == 0 || nbc == 0) return orc_merkle_root(NULL, 0, F, root);
    uint64_t nlr = (nbc + G - 1) / G, nl = n_rows * nlr;
    uint8_t *leaves = (uint8_t *)malloc(32 * nl);
    for (uint64_t r = 0; r < n_rows; r++)
        for (uint64_t g = 0; g < nlr; g++) {
            uint64_t b0 = g * G, b1 = b0 + G < nbc ? b0 + G : nbc;
            orc_sha256(bytes + (r * nbc + b0) * per_block, (b1 - b0) * per_block, leaves + 32 * (r * nlr + g));
        }
    int rc = orc_merkle_root(leaves, nl, F, root);
    free(leaves);
    return rc;
}

/* ------------------------------------------------------------------------------------------ */
/* AES-128 — FIPS-197                                                                          */
/* ------------------------------------------------------------------------------------------ */

static uint8_t xtime(uint8_t a) { return (uint8_t)((a << 1) ^ ((a & 0x80) ? 0x1b : 0x00)); } /* FIPS-197 4.2.1 */

static uint8_t gf_mul(uint8_t a, uint8_t b) { /* FIPS-197 4.2: multiplication modulo x^8+x^4+x^3+x+1 */
    uint8_t p = 0;
    for (int i = 0; i < 8; i++) { if (b & 1) p ^= a; a = xtime(a); b >>= 1; }
    return p;
}

static uint8_t gf_inv(uint8_t a) { /* a^254 = a^-1 in GF(2^8); 0 -> 0 (FIPS-197 5.1.1 step 1) */
    if (a == 0) return 0;
    uint8_t r = 1;
    for (int i = 0; i < 254; i++) r = gf_mul(r, a);
    return r;
}

static uint8_t sbox(uint8_t x) { /* FIPS-197 5.1.1: inverse, then affine transformation with c = 0x63 */
    uint8_t b = gf_inv(x), r = 0;
    for (int i = 0; i < 8; i++) {
        int bit = ((b >> i) ^ (b >> ((i + 4) & 7)) ^ (b >> ((i + 5) & 7)) ^ (b >> ((i + 6) & 7)) ^ (b >> ((i + 7) & 7)) ^
                   (0x63 >> i)) & 1;
        r |= (uint8_t)(bit << i);
    }
    return r;
}

static uint8_t SBOX[256];
static int SBOX_ready = 0;
static void sbox_init(void) {
    if (!SBOX_ready) { for (int i = 0; i < 256; i++) SBOX[i] = sbox((uint8_t)i); SBOX_ready = 1; }
}
void orc_aes_sbox(uint8_t out[256]) { sbox_init(); memcpy(out, SBOX, 256); }

/* FIPS-197 5.2 KeyExpansion, Nk = 4, Nr = 10: 11 round keys of 16 bytes, column-major as the state */
void orc_aes128_expand_key(const uint8_t key[16], uint8_t rk[176]) {
    sbox_init();
    memcpy(rk, key, 16);
    uint8_t rcon = 0x01;
    for (int i = 4; i < 44; i++) {
        uint8_t t[4];
        memcpy(t, rk + 4 * (i - 1), 4);
        if (i % 4 == 0) {
            uint8_t t0 = t[0]; /* RotWord */
            t[0] = SBOX[t[1]] ^ rcon; t[1] = SBOX[t[2]]; t[2] = SBOX[t[3]]; t[3] = SBOX[t0]; /* SubWord ^ Rcon */
            rcon = xtime(rcon);
        }
        for (int j = 0; j < 4; j++) rk[4 * i + j] = rk[4 * (i - 4) + j] ^ t[j];
    }
}

/* FIPS-197 5.1 Cipher. State s[r + 4c] = in[r + 4c] (3.4). */
void orc_aes128_encrypt_block(const uint8_t rk[176], const uint8_t in[16], uint8_t out[16]) {
    uint8_t s[16], t[16];
    sbox_init();
    for (int i = 0; i < 16; i++) s[i] = in[i] ^ rk[i]; /* AddRoundKey(0) */
    for (int round = 1; round <= 10; round++) {
        for (int i = 0; i < 16; i++) s[i] = SBOX[s[i]];                                   /* SubBytes */
        for (int c = 0; c < 4; c++)                                                         /* ShiftRows: row r left by r */
            for (int r = 0; r < 4; r++) t[r + 4 * c] = s[r + 4 * ((c + r) & 3)];
        if (round != 10) {                                                                  /* MixColumns 5.1.3 */
            for (int c = 0; c < 4; c++) {
                uint8_t a0 = t[4 * c], a1 = t[4 * c + 1], a2 = t[4 * c + 2], a3 = t[4 * c + 3];
                s[4 * c + 0] = (uint8_t)(xtime(a0) ^ (xtime(a1) ^ a1) ^ a2 ^ a3);
                s[4 * c + 1] = (uint8_t)(a0 ^ xtime(a1) ^ (xtime(a2) ^ a2) ^ a3);
                s[4 * c + 2] = (uint8_t)(a0 ^ a1 ^ xtime(a2) ^ (xtime(a3) ^ a3));
                s[4 * c + 3] = (uint8_t)((xtime(a0) ^ a0) ^ a1 ^ a2 ^ xtime(a3));
            }
        } else memcpy(s, t, 16);
        for (int i = 0; i < 16; i++) s[i] ^= rk[16 * round + i];                            /* AddRoundKey */
    }
    memcpy(out, s, 16);
}

/* SP 800-38A 6.5 CTR with the standard incrementing function over all 128 bits (B.1, m = 128):
 * T_i = (nonce + i) mod 2^128, big-endian; buf[16 i .. 16 i + 15] ^= AES_K(T_i); a partial last block
 * uses the leading bytes of the keystream block. `first_block` lets a caller address a sub-range. */
void orc_aes128_ctr_xor(const uint8_t key[16], const uint8_t nonce[16], uint64_t first_block, uint8_t *buf, uint64_t n) {
    uint8_t rk[176], ctr[16], ks[16];
    orc_aes128_expand_key(key, rk);
    uint64_t nblocks = (n + 15) / 16;
    for (uint64_t i = 0; i < nblocks; i++) {
        /* ctr = nonce + (first_block + i), 128-bit big-endian addition */
        uint64_t add = first_block + i;
        unsigned carry = 0;
        for (int j = 15; j >= 0; j--) {
            unsigned a = (j >= 8) ? (unsigned)((add >> (8 * (15 - j))) & 0xff) : 0u;
            unsigned v = nonce[j] + a + carry;
            ctr[j] = (uint8_t)v; carry = v >> 8;
        }
        orc_aes128_encrypt_block(rk, ctr, ks);
        uint64_t lo = 16 * i, hi = lo + 16 < n ? lo + 16 : n;
        for (uint64_t p = lo; p < hi; p++) buf[p] ^= ks[p - lo];
    }
}

/* ------------------------------------------------------------------------------------------ */
/* DCT 8x8 — the defining double sum, orthonormal scaling                   */
/* ------------------------------------------------------------------------------------------ */

static const double PI = 3.14159265358979323846264338327950288;

/* X[u][v] = 1/4 C(u) C(v) sum_i sum_j x[i][j] cos((2i+1) u pi/16) cos((2j+1) v pi/16); u: rows (vertical) */
void orc_dct8x8(const double x[64], double X[64]) {
    for (int u = 0; u < 8; u++)
        for (int v = 0; v < 8; v++) {
            double sum = 0.0;
            for (int i = 0; i < 8; i++)
                for (int j = 0; j < 8; j++)
                    sum += x[8 * i + j] * cos((2 * i + 1) * u * PI / 16.0) * cos((2 * j + 1) * v * PI / 16.0);
            double cu = (u == 0) ? sqrt(0.5) : 1.0, cv = (v == 0) ? sqrt(0.5) : 1.0;
            X[8 * u + v] = 0.25 * cu * cv * sum;
        }
}

/* x[i][j] = 1/4 sum_u sum_v C(u) C(v) X[u][v] cos((2i+1) u pi/16) cos((2j+1) v pi/16) */
void orc_idct8x8(const double X[64], double x[64]) {
    for (int i = 0; i < 8; i++)
        for (int j = 0; j < 8; j++) {
            double sum = 0.0;
            for (int u = 0; u < 8; u++)
                for (int v = 0; v < 8; v++) {
                    double cu = (u == 0) ? sqrt(0.5) : 1.0, cv = (v == 0) ? sqrt(0.5) : 1.0;
                    sum += cu * cv * X[8 * u + v] * cos((2 * i + 1) * u * PI / 16.0) * cos((2 * j + 1) * v * PI / 16.0);
                }
            x[8 * i + j] = 0.25 * sum;
        }
}

/* zigzag index z -> (row, col): anti-diagonals s = row + col = 0..14; even s: row descending, odd s:
 * row ascending. z = 0..5 gives [0,0],[0,1],[1,0],[2,0],[1,1],[0,2] = P:494's default selection. */
int orc_zigzag(int z, int *row, int *col) {
    if (z < 0 || z > 63) return -1;
    int idx = 0;
    for (int s = 0; s <= 14; s++) {
        int rlo = s > 7 ? s - 7 : 0, rhi = s < 7 ? s : 7;
        if (s % 2 == 0) {
            for (int r = rhi; r >= rlo; r--, idx++) if (idx == z) { *row = r; *col = s - r; return 0; }
        } else {
            for (int r = rlo; r <= rhi; r++, idx++) if (idx == z) { *row = r; *col = s - r; return 0; }
        }
    }
    return -1;
}

static int check_dct_dims(int w, int h, int c, int k) {
    if (w <= 0 || h <= 0 || (w % 8) || (h % 8)) return -1;
    if (!(c == 1 || c == 3 || c == 4)) return -2;
    if (k < 0 || k > 63) return -2;
    return 0;
}

/* Steps 1-2 of the path + zigzag reorder: image uint8[H][W][C] -> coef double[b][z], b = (c*nbr+br)*nbc+bc,
 * z = zigzag index. No level shift. */
int orc_dct_coefficients(const uint8_t *image, int w, int h, int c, double *coef) {
    if (check_dct_dims(w, h, c, 0)) return -1;
    int nbr = h / 8, nbc = w / 8;
    for (int ch = 0; ch < c; ch++)
        for (int br = 0; br < nbr; br++)
            for (int bc = 0; bc < nbc; bc++) {
                double x[64], X[64];
                for (int i = 0; i < 8; i++)
                    for (int j = 0; j < 8; j++)
                        x[8 * i + j] = (double)image[((size_t)(8 * br + i) * w + (8 * bc + j)) * c + ch];
                orc_dct8x8(x, X);
                size_t b = ((size_t)ch * nbr + br) * nbc + bc;
                for (int z = 0; z < 64; z++) {
                    int r, q;
                    orc_zigzag(z, &r, &q);
                    coef[64 * b + z] = X[8 * r + q];
                }
            }
    return 0;
}

static void put_f32le(uint8_t *p, float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    p[0] = (uint8_t)u; p[1] = (uint8_t)(u >> 8); p[2] = (uint8_t)(u >> 16); p[3] = (uint8_t)(u >> 24);
}
static float get_f32le(const uint8_t *p) {
    uint32_t u = (uint32_t)p[0] | ((uint32_t)p[1] << 8) | ((uint32_t)p[2] << 16) | ((uint32_t)p[3] << 24);
    float f;
    memcpy(&f, &u, 4);
    return f;
}

/* Steps 3-5 given float32 coefficients coef32[b][z] (zigzag order): select/pack, AES-CTR on private,
 * Merkle digests of the stored bytes. This is what stage-(ii) parity feeds the GPU's own coefficient bytes to. */
int orc_fragment_from_coef32(const float *coef32, int w, int h, int c, int k, const uint8_t key[16],
                             const uint8_t nonce[16], int G, int F, uint8_t *priv, uint8_t *pub, uint8_t digests[64]) {
    if (check_dct_dims(w, h, c, k)) return -1;
    size_t nb = (size_t)c * (h / 8) * (w / 8);
    int P = k + 1, Q = 63 - k;
    for (size_t b = 0; b < nb; b++) {
        for (int z = 0; z <= k; z++) put_f32le(priv + 4 * (b * P + z), coef32[64 * b + z]);
        for (int z = k + 1; z < 64; z++) put_f32le(pub + 4 * (b * Q + (z - k - 1)), coef32[64 * b + z]);
    }
    orc_aes128_ctr_xor(key, nonce, 0, priv, 4 * nb * P);
    int rc = orc_merkle_blocks(priv, (uint64_t)c * (h / 8), (uint64_t)(w / 8), 4 * (uint64_t)P, G, F, digests);
    if (rc) return rc;
    return orc_merkle_blocks(pub, (uint64_t)c * (h / 8), (uint64_t)(w / 8), 4 * (uint64_t)Q, G, F, digests + 32);
}

/* Whole forward path: image -> private (ciphertext), public, digests. Double DCT rounded to float32 (RNE). */
int orc_fragment_dct(const uint8_t *image, int w, int h, int c, int k, const uint8_t key[16], const uint8_t nonce[16],
                     int G, int F, uint8_t *priv, uint8_t *pub, uint8_t digests[64]) {
    if (check_dct_dims(w, h, c, k)) return -1;
    size_t nb = (size_t)c * (h / 8) * (w / 8);
    double *coef = (double *)malloc(sizeof(double) * 64 * nb);
    float *c32 = (float *)malloc(sizeof(float) * 64 * nb);
    if (!coef || !c32) { free(coef); free(c32); return -3; }
    orc_dct_coefficients(image, w, h, c, coef);
    for (size_t i = 0; i < 64 * nb; i++) c32[i] = (float)coef[i];
    int rc = orc_fragment_from_coef32(c32, w, h, c, k, key, nonce, G, F, priv, pub, digests);
    free(coef); free(c32);
    return rc;
}

/* Inverse path (steps 6-8): verify (flags bit0 private mismatch, bit1 public mismatch; skipped when
 * expected == NULL), decrypt, merge, IDCT by the defining sum, round to nearest even (lrint under the
 * default rounding mode), clamp to [0,255]. The image is written regardless of the flags (A10). */
int orc_defragment_dct(const uint8_t *priv, const uint8_t *pub, int w, int h, int c, int k, const uint8_t key[16],
                       const uint8_t nonce[16], int G, int F, const uint8_t *expected /* 64 B or NULL */,
                       uint8_t *image_out, uint32_t *flags) {
    if (check_dct_dims(w, h, c, k)) return -1;
    int nbr = h / 8, nbc = w / 8, P = k + 1, Q = 63 - k;
    size_t nb = (size_t)c * nbr * nbc;
    if (flags) *flags = 0;
    if (expected) {
        uint8_t dg[64];
        orc_merkle_blocks(priv, (uint64_t)c * nbr, (uint64_t)nbc, 4 * (uint64_t)P, G, F, dg);
        orc_merkle_blocks(pub, (uint64_t)c * nbr, (uint64_t)nbc, 4 * (uint64_t)Q, G, F, dg + 32);
        uint32_t fl = 0;
        if (memcmp(dg, expected, 32)) fl |= 1u;
        if (memcmp(dg + 32, expected + 32, 32)) fl |= 2u;
        if (flags) *flags = fl;
    }
    uint8_t *pt = (uint8_t *)malloc(4 * nb * P);
    if (!pt) return -3;
    memcpy(pt, priv, 4 * nb * P);
    orc_aes128_ctr_xor(key, nonce, 0, pt, 4 * nb * P); /* CTR is its own inverse */
    for (int ch = 0; ch < c; ch++)
        for (int br = 0; br < nbr; br++)
            for (int bc = 0; bc < nbc; bc++) {
                size_t b = ((size_t)ch * nbr + br) * nbc + bc;
                double X[64], x[64];
                for (int z = 0; z < 64; z++) {
                    int r, q;
                    orc_zigzag(z, &r, &q);
                    float f = (z <= k) ? get_f32le(pt + 4 * (b * P + z)) : get_f32le(pub + 4 * (b * Q + (z - k - 1)));
                    X[8 * r + q] = (double)f;
                }
                orc_idct8x8(X, x);
                for (int i = 0; i < 8; i++)
                    for (int j = 0; j < 8; j++) {
                        double v = x[8 * i + j];
                        long q = (v != v) ? 0 : (v > 1e9 ? 1000000000L : (v < -1e9 ? -1000000000L : lrint(v)));
                        if (q < 0) q = 0;
                        if (q > 255) q = 255;
                        image_out[((size_t)(8 * br + i) * w + (8 * bc + j)) * c + ch] = (uint8_t)q;
                    }
            }
    free(pt);
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* Le Gall 5/3 integer lifting DWT (A12-A16)                               */
/* ------------------------------------------------------------------------------------------ */

static int32_t floor_div(int32_t a, int32_t b) { /* floor(a / b), b > 0: "largest integer not exceeding a" */
    int32_t q = a / b, r = a % b;
    return (r != 0 && r < 0) ? q - 1 : q;
}

/* 1-D analysis of x[0..N), N even, stride-addressed; output s[0..N/2) then d[0..N/2) into y[0..N). */
void orc_dwt53_fwd_1d(const int32_t *x, int N, int32_t *y) {
    int half = N / 2;
    int32_t *s = y, *d = y + half;
    for (int n = 0; n < half; n++) { /* eq. (1): predict */
        int32_t right = (2 * n + 2 < N) ? x[2 * n + 2] : x[N - 2]; /* x_ext(N) = x(N-2) */
        d[n] = x[2 * n + 1] - floor_div(x[2 * n] + right, 2);
    }
    for (int n = 0; n < half; n++) { /* eq. (2), A12 reading: update from the high-pass outputs */
        int32_t left = (n > 0) ? d[n - 1] : d[0]; /* y_ext(-1) = y(1) */
        s[n] = x[2 * n] + floor_div(left + d[n] + 2, 4);
    }
}

/* 1-D synthesis: y = [s | d] -> x, undoing the update then the predict (P:822 exact inverse). */
void orc_dwt53_inv_1d(const int32_t *y, int N, int32_t *x) {
    int half = N / 2;
    const int32_t *s = y, *d = y + half;
    for (int n = 0; n < half; n++) {
        int32_t left = (n > 0) ? d[n - 1] : d[0];
        x[2 * n] = s[n] - floor_div(left + d[n] + 2, 4);
    }
    for (int n = 0; n < half; n++) {
        int32_t right = (2 * n + 2 < N) ? x[2 * n + 2] : x[N - 2];
        x[2 * n + 1] = d[n] + floor_div(x[2 * n] + right, 2);
    }
}

static int check_dwt_dims(int w, int h, int c, int L) {
    if (w <= 0 || h <= 0) return -1;
    if (!(c == 1 || c == 3 || c == 4)) return -2;
    if (L < 1 || L > 6) return -2;
    if ((w % (1 << L)) || (h % (1 << L))) return -1;
    return 0;
}

/* In-place L-level 2-D transform of one int32 plane p[h][w] (Mallat layout: LL_L top-left). Rows first,
 * then columns. Returns -4 if any coefficient leaves the int16 range (A16). */
int orc_dwt53_fwd_plane(int32_t *p, int w, int h, int L) {
    int32_t *line = (int32_t *)malloc(sizeof(int32_t) * (size_t)(w > h ? w : h) * 2);
    int32_t *out = line + (w > h ? w : h);
    for (int l = 0; l < L; l++) {
        int cw = w >> l, chh = h >> l;
        for (int r = 0; r < chh; r++) { /* horizontal */
            for (int i = 0; i < cw; i++) line[i] = p[(size_t)r * w + i];
            orc_dwt53_fwd_1d(line, cw, out);
            for (int i = 0; i < cw; i++) p[(size_t)r * w + i] = out[i];
        }
        for (int q = 0; q < cw; q++) { /* vertical */
            for (int i = 0; i < chh; i++) line[i] = p[(size_t)i * w + q];
            orc_dwt53_fwd_1d(line, chh, out);
            for (int i = 0; i < chh; i++) p[(size_t)i * w + q] = out[i];
        }
    }
    free(line);
    for (size_t i = 0; i < (size_t)w * h; i++) if (p[i] < -32768 || p[i] > 32767) return -4;
    return 0;
}

int orc_dwt53_inv_plane(int32_t *p, int w, int h, int L) {
    int32_t *line = (int32_t *)malloc(sizeof(int32_t) * (size_t)(w > h ? w : h) * 2);
    int32_t *out = line + (w > h ? w : h);
    for (int l = L - 1; l >= 0; l--) {
        int cw = w >> l, chh = h >> l;
        for (int q = 0; q < cw; q++) { /* vertical first (reverse of the forward order) */
            for (int i = 0; i < chh; i++) line[i] = p[(size_t)i * w + q];
            orc_dwt53_inv_1d(line, chh, out);
            for (int i = 0; i < chh; i++) p[(size_t)i * w + q] = out[i];
        }
        for (int r = 0; r < chh; r++) {
            for (int i = 0; i < cw; i++) line[i] = p[(size_t)r * w + i];
            orc_dwt53_inv_1d(line, cw, out);
            for (int i = 0; i < cw; i++) p[(size_t)r * w + i] = out[i];
        }
    }
    free(line);
    return 0;
}

static void put_i16le(uint8_t *p, int32_t v) { uint16_t u = (uint16_t)(int16_t)v; p[0] = (uint8_t)u; p[1] = (uint8_t)(u >> 8); }
static int32_t get_i16le(const uint8_t *p) { return (int32_t)(int16_t)((uint16_t)p[0] | ((uint16_t)p[1] << 8)); }

/* Rectangle of band `band` (0 = HL top-right, 1 = LH bottom-left, 2 = HH bottom-right) at level l (1-based)
 * inside the Mallat plane: origin (r0, c0), size (h>>l) x (w>>l). */
static void band_origin(int w, int h, int l, int band, int *r0, int *c0) {
    int bw = w >> l, bh = h >> l;
    *r0 = (band == 0) ? 0 : bh;
    *c0 = (band == 1) ? 0 : bw;
}

/* DWT forward path D1-D5: image -> private (LL_L under AES-CTR), public (other subbands), digests. */
int orc_fragment_dwt(const uint8_t *image, int w, int h, int c, int L, const uint8_t key[16], const uint8_t nonce[16],
                     uint64_t leaf_bytes, int F, uint8_t *priv, uint8_t *pub, uint8_t digests[64]) {
    if (check_dwt_dims(w, h, c, L)) return -1;
    int lw = w >> L, lh = h >> L;
    size_t priv_per_c = (size_t)lw * lh * 2, pub_per_c = ((size_t)w * h - (size_t)lw * lh) * 2;
    int32_t *p = (int32_t *)malloc(sizeof(int32_t) * (size_t)w * h);
    if (!p) return -3;
    for (int ch = 0; ch < c; ch++) {
        for (int y = 0; y < h; y++)
            for (int x = 0; x < w; x++) p[(size_t)y * w + x] = (int32_t)image[((size_t)y * w + x) * c + ch] - 128;
        int rc = orc_dwt53_fwd_plane(p, w, h, L);
        if (rc) { free(p); return rc; }
        uint8_t *o = priv + ch * priv_per_c;
        for (int y = 0; y < lh; y++)
            for (int x = 0; x < lw; x++, o += 2) put_i16le(o, p[(size_t)y * w + x]);
        o = pub + ch * pub_per_c;
        for (int l = L; l >= 1; l--)
            for (int band = 0; band < 3; band++) {
                int r0, c0, bw = w >> l, bh = h >> l;
                band_origin(w, h, l, band, &r0, &c0);
                for (int y = 0; y < bh; y++)
                    for (int x = 0; x < bw; x++, o += 2) put_i16le(o, p[(size_t)(r0 + y) * w + (c0 + x)]);
            }
    }
    free(p);
    orc_aes128_ctr_xor(key, nonce, 0, priv, priv_per_c * c);
    int rc = orc_merkle_stream(priv, priv_per_c * c, leaf_bytes, F, digests);
    if (rc) return rc;
    return orc_merkle_stream(pub, pub_per_c * c, leaf_bytes, F, digests + 32);
}

/* Plain (unencrypted) coefficient planes, for coefficient-level tests: out int32[c][h][w] Mallat layout. */
int orc_dwt_coefficients(const uint8_t *image, int w, int h, int c, int L, int32_t *out) {
    if (check_dwt_dims(w, h, c, L)) return -1;
    for (int ch = 0; ch < c; ch++) {
        int32_t *p = out + (size_t)ch * w * h;
        for (int y = 0; y < h; y++)
            for (int x = 0; x < w; x++) p[(size_t)y * w + x] = (int32_t)image[((size_t)y * w + x) * c + ch] - 128;
        int rc = orc_dwt53_fwd_plane(p, w, h, L);
        if (rc) return rc;
    }
    return 0;
}

/* DWT inverse path D6-D8. +128, clamp to [0,255] (exact on untampered data). */
int orc_defragment_dwt(const uint8_t *priv, const uint8_t *pub, int w, int h, int c, int L, const uint8_t key[16],
                       const uint8_t nonce[16], uint64_t leaf_bytes, int F, const uint8_t *expected,
                       uint8_t *image_out, uint32_t *flags) {
    if (check_dwt_dims(w, h, c, L)) return -1;
    int lw = w >> L, lh = h >> L;
    size_t priv_per_c = (size_t)lw * lh * 2, pub_per_c = ((size_t)w * h - (size_t)lw * lh) * 2;
    if (flags) *flags = 0;
    if (expected) {
        uint8_t dg[64];
        orc_merkle_stream(priv, priv_per_c * c, leaf_bytes, F, dg);
        orc_merkle_stream(pub, pub_per_c * c, leaf_bytes, F, dg + 32);
        uint32_t fl = 0;
        if (memcmp(dg, expected, 32)) fl |= 1u;
        if (memcmp(dg + 32, expected + 32, 32)) fl |= 2u;
        if (flags) *flags = fl;
    }
    uint8_t *pt = (uint8_t *)malloc(priv_per_c * c);
    int32_t *p = (int32_t *)malloc(sizeof(int32_t) * (size_t)w * h);
    if (!pt || !p) { free(pt); free(p); return -3; }
    memcpy(pt, priv, priv_per_c * c);
    orc_aes128_ctr_xor(key, nonce, 0, pt, priv_per_c * c);
    for (int ch = 0; ch < c; ch++) {
        const uint8_t *o = pt + ch * priv_per_c;
        for (int y = 0; y < lh; y++)
            for (int x = 0; x < lw; x++, o += 2) p[(size_t)y * w + x] = get_i16le(o);
        o = pub + ch * pub_per_c;
        for (int l = L; l >= 1; l--)
            for (int band = 0; band < 3; band++) {
                int r0, c0, bw = w >> l, bh = h >> l;
                band_origin(w, h, l, band, &r0, &c0);
                for (int y = 0; y < bh; y++)
                    for (int x = 0; x < bw; x++, o += 2) p[(size_t)(r0 + y) * w + (c0 + x)] = get_i16le(o);
            }
        orc_dwt53_inv_plane(p, w, h, L);
        for (int y = 0; y < h; y++)
            for (int x = 0; x < w; x++) {
                int32_t v = p[(size_t)y * w + x] + 128;
                if (v < 0) v = 0;
                if (v > 255) v = 255;
                image_out[((size_t)y * w + x) * c + ch] = (uint8_t)v;
            }
    }
    free(pt); free(p);
    return 0;
}
