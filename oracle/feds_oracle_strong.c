/*
 * feds_oracle_strong.c — CPU ORACLE for the report's STRONG level of protection (section 6.3.2, P:502-516,
 * Figure 8; timings P:676-692). TEST INFRASTRUCTURE, NOT PRODUCT (see feds_oracle.c); shares nothing with the CUDA path.
 *
 * What the report says: Part 1 (the selected low frequencies of a block) is encrypted as in the first level; "the
 * reverse DCT result of the rest DCT coefficients padded with zero contains 64 pixels storing in byte which is exactly 512 bits";
 * SHA-512 of the selected coefficients gives a 512-bit string, and "the XOR step can protect every pixel block by block".
 * Where it is silent, DESIGN.md section 2.3 fixes (readings S1-S5):
 *   S1  the remainder in bytes. By linearity IDCT(rest padded with zeros) = x - IDCT(Part 1 padded with zeros); it is zero-mean and
 *       can reach +-255, so it does not fit a byte as a number. It is stored modulo 256, and the low-pass image is computed in
 *       exact integer arithmetic from the STORED float32 coefficients, so that both directions -- and any two implementations --
 *       obtain the same bytes:  q_z = rne(8 c_z) (saturated to int32, NaN -> 0),  B[z][p] = rne(4096 b_z(p)) with b_z the
 *       orthonormal 8x8 DCT basis function of zigzag index z at pixel p = 8 i + j,
 *       L[p] = floor((sum_{z<=k} q_z B[z][p] + 2^14) / 2^15),   r[p] = (x[p] - L[p]) mod 256.
 *       |(x - L) - IDCT(rest)| <= 1 (pinned against scipy in tests/test_oracle_strong.py).
 *   S2  SHA-512 input: the block's Part 1 as stored before encryption: 4 (k + 1) bytes, float32 little-endian, zigzag order.
 *   S3  keystream byte p = byte p of the digest (H0 .. H7 big-endian, FIPS 180-4 6.4.2 step 4), XORed with r[p], p = 8 i + j.
 *   S4  public fragment: uint8 [block][p], 64 bytes per block, block order as DESIGN.md 2.1; private fragment as 2.1.
 *   S5  digests: the Merkle layout of 2.1 over the stored bytes (public leaf = 8 blocks x 64 bytes).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* from feds_oracle.c */
int orc_zigzag(int z, int *row, int *col);
int orc_dct_coefficients(const uint8_t *image, int w, int h, int c, double *coef);
void orc_aes128_ctr_xor(const uint8_t key[16], const uint8_t nonce[16], uint64_t first_block, uint8_t *buf, uint64_t n);
int orc_merkle_blocks(const uint8_t *bytes, uint64_t n_rows, uint64_t nbc, uint64_t per_block, int G, int F, uint8_t root[32]);

/* ------------------------------------------------------------------------------------------ */
/* SHA-512 — FIPS 180-4 section 6.4                                                             */
/* ------------------------------------------------------------------------------------------ */
static uint64_t rotr64(uint64_t x, int n) { return (x >> n) | (x << (64 - n)); }

/* FIPS 180-4 4.2.3: first 64 bits of the fractional parts of the cube roots of the first 80 primes */
static const uint64_t SHA512_K[80] = {
    0x428a2f98d728ae22ULL, 0x7137449123ef65cdULL, 0xb5c0fbcfec4d3b2fULL, 0xe9b5dba58189dbbcULL, 0x3956c25bf348b538ULL,
    0x59f111f1b605d019ULL, 0x923f82a4af194f9bULL, 0xab1c5ed5da6d8118ULL, 0xd807aa98a3030242ULL, 0x12835b0145706fbeULL,
    0x243185be4ee4b28cULL, 0x550c7dc3d5ffb4e2ULL, 0x72be5d74f27b896fULL, 0x80deb1fe3b1696b1ULL, 0x9bdc06a725c71235ULL,
    0xc19bf174cf692694ULL, 0xe49b69c19ef14ad2ULL, 0xefbe4786384f25e3ULL, 0x0fc19dc68b8cd5b5ULL, 0x240ca1cc77ac9c65ULL,
    0x2de92c6f592b0275ULL, 0x4a7484aa6ea6e483ULL, 0x5cb0a9dcbd41fbd4ULL, 0x76f988da831153b5ULL, 0x983e5152ee66dfabULL,
    0xa831c66d2db43210ULL, 0xb00327c898fb213fULL, 0xbf597fc7beef0ee4ULL, 0xc6e00bf33da88fc2ULL, 0xd5a79147930aa725ULL,
    0x06ca6351e003826fULL, 0x142929670a0e6e70ULL, 0x27b70a8546d22ffcULL, 0x2e1b21385c26c926ULL, 0x4d2c6dfc5ac42aedULL,
    0x53380d139d95b3dfULL, 0x650a73548baf63deULL, 0x766a0abb3c77b2a8ULL, 0x81c2c92e47edaee6ULL, 0x92722c851482353bULL,
    0xa2bfe8a14cf10364ULL, 0xa81a664bbc423001ULL, 0xc24b8b70d0f89791ULL, 0xc76c51a30654be30ULL, 0xd192e819d6ef5218ULL,
    0xd69906245565a910ULL, 0xf40e35855771202aULL, 0x106aa07032bbd1b8ULL, 0x19a4c116b8d2d0c8ULL, 0x1e376c085141ab53ULL,
    0x2748774cdf8eeb99ULL, 0x34b0bcb5e19b48a8ULL, 0x391c0cb3c5c95a63ULL, 0x4ed8aa4ae3418acbULL, 0x5b9cca4f7763e373ULL,
    0x682e6ff3d6b2b8a3ULL, 0x748f82ee5defb2fcULL, 0x78a5636f43172f60ULL, 0x84c87814a1f0ab72ULL, 0x8cc702081a6439ecULL,
    0x90befffa23631e28ULL, 0xa4506cebde82bde9ULL, 0xbef9a3f7b2c67915ULL, 0xc67178f2e372532bULL, 0xca273eceea26619cULL,
    0xd186b8c721c0c207ULL, 0xeada7dd6cde0eb1eULL, 0xf57d4f7fee6ed178ULL, 0x06f067aa72176fbaULL, 0x0a637dc5a2c898a6ULL,
    0x113f9804bef90daeULL, 0x1b710b35131c471bULL, 0x28db77f523047d84ULL, 0x32caab7b40c72493ULL, 0x3c9ebe0a15c9bebcULL,
    0x431d67c49c100d4cULL, 0x4cc5d4becb3e42b6ULL, 0x597f299cfc657e2aULL, 0x5fcb6fab3ad6faecULL, 0x6c44198c4a475817ULL};

static void sha512_block(uint64_t H[8], const uint8_t M[128]) {
    uint64_t W[80];
    for (int t = 0; t < 16; t++) {
        uint64_t v = 0;
        for (int b = 0; b < 8; b++) v = (v << 8) | M[8 * t + b];
        W[t] = v;
    }
    for (int t = 16; t < 80; t++) {
        uint64_t s0 = rotr64(W[t - 15], 1) ^ rotr64(W[t - 15], 8) ^ (W[t - 15] >> 7);   /* sigma0, eq. 4.12 */
        uint64_t s1 = rotr64(W[t - 2], 19) ^ rotr64(W[t - 2], 61) ^ (W[t - 2] >> 6);     /* sigma1, eq. 4.13 */
        W[t] = s1 + W[t - 7] + s0 + W[t - 16];
    }
    uint64_t a = H[0], b = H[1], c = H[2], d = H[3], e = H[4], f = H[5], g = H[6], h = H[7];
    for (int t = 0; t < 80; t++) {
        uint64_t S1 = rotr64(e, 14) ^ rotr64(e, 18) ^ rotr64(e, 41);   /* Sigma1, eq. 4.11 */
        uint64_t ch = (e & f) ^ (~e & g);
        uint64_t T1 = h + S1 + ch + SHA512_K[t] + W[t];
        uint64_t S0 = rotr64(a, 28) ^ rotr64(a, 34) ^ rotr64(a, 39);   /* Sigma0, eq. 4.10 */
        uint64_t maj = (a & b) ^ (a & c) ^ (b & c);
        uint64_t T2 = S0 + maj;
        h = g; g = f; f = e; e = d + T1; d = c; c = b; b = a; a = T1 + T2;
    }
    H[0] += a; H[1] += b; H[2] += c; H[3] += d; H[4] += e; H[5] += f; H[6] += g; H[7] += h;
}

void orc_sha512(const uint8_t *msg, uint64_t n, uint8_t out[64]) {
    uint64_t H[8] = {0x6a09e667f3bcc908ULL, 0xbb67ae8584caa73bULL, 0x3c6ef372fe94f82bULL, 0xa54ff53a5f1d36f1ULL,
                     0x510e527fade682d1ULL, 0x9b05688c2b3e6c1fULL, 0x1f83d9abfb41bd6bULL, 0x5be0cd19137e2179ULL};   /* 5.3.5 */
    uint64_t full = n / 128;
    for (uint64_t i = 0; i < full; i++) sha512_block(H, msg + 128 * i);
    uint8_t tail[256];
    uint64_t rem = n - 128 * full;
    memset(tail, 0, sizeof tail);
    if (rem) memcpy(tail, msg + 128 * full, rem);
    tail[rem] = 0x80;                                   /* 5.1.2: bit "1", then zeros, then the 128-bit length in bits */
    int blocks = (rem + 1 + 16 <= 128) ? 1 : 2;
    uint64_t bits = n * 8;                              /* n < 2^61 */
    for (int b = 0; b < 8; b++) tail[128 * blocks - 1 - b] = (uint8_t)(bits >> (8 * b));
    for (int i = 0; i < blocks; i++) sha512_block(H, tail + 128 * i);
    for (int i = 0; i < 8; i++)
        for (int b = 0; b < 8; b++) out[8 * i + b] = (uint8_t)(H[i] >> (56 - 8 * b));
}

/* ------------------------------------------------------------------------------------------ */
/* strong level: DESIGN.md 2.3                                                                  */
/* ------------------------------------------------------------------------------------------ */
static const double PI = 3.14159265358979323846264338327950288;

/* B[z][p] = rne(4096 * b_z(p)),  b_z(8i+j) = 1/4 C(u) C(v) cos((2i+1) u pi/16) cos((2j+1) v pi/16),  (u, v) = zigzag(z) */
void orc_strong_basis(int32_t B[64 * 64]) {
    for (int z = 0; z < 64; z++) {
        int u, v;
        orc_zigzag(z, &u, &v);
        double cu = u ? 1.0 : sqrt(0.5), cv = v ? 1.0 : sqrt(0.5);
        for (int i = 0; i < 8; i++)
            for (int j = 0; j < 8; j++)
                B[64 * z + 8 * i + j] = (int32_t)lrint(4096.0 * 0.25 * cu * cv * cos((2 * i + 1) * u * PI / 16.0) * cos((2 * j + 1) * v * PI / 16.0));
    }
}

static float get_f32le(const uint8_t *p) {
    uint32_t u = (uint32_t)p[0] | ((uint32_t)p[1] << 8) | ((uint32_t)p[2] << 16) | ((uint32_t)p[3] << 24);
    float f;
    memcpy(&f, &u, 4);
    return f;
}
static void put_f32le(uint8_t *p, float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    p[0] = (uint8_t)u; p[1] = (uint8_t)(u >> 8); p[2] = (uint8_t)(u >> 16); p[3] = (uint8_t)(u >> 24);
}

/* q = rne(8 c), saturated to the int32 range, NaN -> 0 (S1) */
static int64_t quantise8(float c) {
    double v = 8.0 * (double)c;
    if (v != v) return 0;
    if (v >= 2147483647.0) return 2147483647LL;
    if (v <= -2147483648.0) return -2147483648LL;
    return (int64_t)lrint(v);
}

/* L[p] mod 256 of one block from its k + 1 plaintext private coefficients (S1). Arithmetic in Z: int64 is exact here. */
static void low_pass_mod256(const int32_t *B, const uint8_t *coef_bytes, int k, uint8_t L[64]) {
    for (int p = 0; p < 64; p++) {
        int64_t acc = 0;
        for (int z = 0; z <= k; z++) acc += quantise8(get_f32le(coef_bytes + 4 * z)) * (int64_t)B[64 * z + p];
        acc += 16384;
        int64_t fl = (acc >= 0) ? (acc >> 15) : -((-acc + 32767) >> 15);   /* floor(acc / 2^15) */
        L[p] = (uint8_t)(fl & 255);
    }
}

static int check_dims(int w, int h, int c, int k) {
    if (w <= 0 || h <= 0 || (w % 8) || (h % 8)) return -1;
    if (!(c == 1 || c == 3 || c == 4)) return -2;
    if (k < 0 || k > 63) return -2;
    return 0;
}

/* Everything after the DCT, given the float32 private coefficients priv32[b][z], z = 0..k (zigzag order): remainder bytes,
 * SHA-512 keystream, XOR, AES-CTR on the private part, Merkle digests. Stage-(ii) parity feeds this the GPU's own decrypted
 * private coefficients. pub: w*h*c bytes. priv: 4 (k+1) bytes per block. */
int orc_fragment_strong_from_priv32(const uint8_t *image, const float *priv32, int w, int h, int c, int k, const uint8_t key[16],
                                    const uint8_t nonce[16], int G, int F, uint8_t *priv, uint8_t *pub, uint8_t digests[64]) {
    if (check_dims(w, h, c, k)) return -1;
    int nbr = h / 8, nbc = w / 8, P = k + 1;
    size_t nb = (size_t)c * nbr * nbc;
    int32_t *B = (int32_t *)malloc(sizeof(int32_t) * 64 * 64);
    if (!B) return -3;
    orc_strong_basis(B);
    for (int ch = 0; ch < c; ch++)
        for (int br = 0; br < nbr; br++)
            for (int bc = 0; bc < nbc; bc++) {
                size_t b = ((size_t)ch * nbr + br) * nbc + bc;
                uint8_t *pc = priv + 4 * b * P;
                for (int z = 0; z <= k; z++) put_f32le(pc + 4 * z, priv32[b * P + z]);
                uint8_t L[64], d[64];
                low_pass_mod256(B, pc, k, L);
                orc_sha512(pc, 4 * (uint64_t)P, d);
                for (int i = 0; i < 8; i++)
                    for (int j = 0; j < 8; j++) {
                        uint8_t x = image[((size_t)(8 * br + i) * w + (8 * bc + j)) * c + ch];
                        pub[64 * b + 8 * i + j] = (uint8_t)((uint8_t)(x - L[8 * i + j]) ^ d[8 * i + j]);
                    }
            }
    free(B);
    orc_aes128_ctr_xor(key, nonce, 0, priv, 4 * nb * P);
    int rc = orc_merkle_blocks(priv, (uint64_t)c * nbr, (uint64_t)nbc, 4 * (uint64_t)P, G, F, digests);
    if (rc) return rc;
    return orc_merkle_blocks(pub, (uint64_t)c * nbr, (uint64_t)nbc, 64, G, F, digests + 32);
}

/* Whole forward path: double DCT (the defining sum), Part 1 rounded to float32, then as above. */
int orc_fragment_dct_strong(const uint8_t *image, int w, int h, int c, int k, const uint8_t key[16], const uint8_t nonce[16], int G,
                            int F, uint8_t *priv, uint8_t *pub, uint8_t digests[64]) {
    if (check_dims(w, h, c, k)) return -1;
    size_t nb = (size_t)c * (h / 8) * (w / 8);
    int P = k + 1;
    double *coef = (double *)malloc(sizeof(double) * 64 * nb);
    float *p32 = (float *)malloc(sizeof(float) * P * nb);
    if (!coef || !p32) { free(coef); free(p32); return -3; }
    orc_dct_coefficients(image, w, h, c, coef);
    for (size_t b = 0; b < nb; b++)
        for (int z = 0; z <= k; z++) p32[b * P + z] = (float)coef[64 * b + z];
    int rc = orc_fragment_strong_from_priv32(image, p32, w, h, c, k, key, nonce, G, F, priv, pub, digests);
    free(coef); free(p32);
    return rc;
}

/* Inverse: verify (optional), decrypt Part 1, rebuild L and the keystream from it, x = ((pub xor d) + L) mod 256. */
int orc_defragment_dct_strong(const uint8_t *priv, const uint8_t *pub, int w, int h, int c, int k, const uint8_t key[16],
                              const uint8_t nonce[16], int G, int F, const uint8_t *expected, uint8_t *image_out, uint32_t *flags) {
    if (check_dims(w, h, c, k)) return -1;
    int nbr = h / 8, nbc = w / 8, P = k + 1;
    size_t nb = (size_t)c * nbr * nbc;
    if (flags) *flags = 0;
    if (expected) {
        uint8_t dg[64];
        orc_merkle_blocks(priv, (uint64_t)c * nbr, (uint64_t)nbc, 4 * (uint64_t)P, G, F, dg);
        orc_merkle_blocks(pub, (uint64_t)c * nbr, (uint64_t)nbc, 64, G, F, dg + 32);
        uint32_t fl = 0;
        if (memcmp(dg, expected, 32)) fl |= 1u;
        if (memcmp(dg + 32, expected + 32, 32)) fl |= 2u;
        if (flags) *flags = fl;
    }
    uint8_t *pt = (uint8_t *)malloc(4 * nb * P);
    int32_t *B = (int32_t *)malloc(sizeof(int32_t) * 64 * 64);
    if (!pt || !B) { free(pt); free(B); return -3; }
    orc_strong_basis(B);
    memcpy(pt, priv, 4 * nb * P);
    orc_aes128_ctr_xor(key, nonce, 0, pt, 4 * nb * P);
    for (int ch = 0; ch < c; ch++)
        for (int br = 0; br < nbr; br++)
            for (int bc = 0; bc < nbc; bc++) {
                size_t b = ((size_t)ch * nbr + br) * nbc + bc;
                uint8_t L[64], d[64];
                low_pass_mod256(B, pt + 4 * b * P, k, L);
                orc_sha512(pt + 4 * b * P, 4 * (uint64_t)P, d);
                for (int i = 0; i < 8; i++)
                    for (int j = 0; j < 8; j++)
                        image_out[((size_t)(8 * br + i) * w + (8 * bc + j)) * c + ch] =
                            (uint8_t)((uint8_t)(pub[64 * b + 8 * i + j] ^ d[8 * i + j]) + L[8 * i + j]);
            }
    free(pt); free(B);
    return 0;
}

/* the signed remainder x - L of every pixel (for the pin against IDCT(rest)): int16 [h][w][c] */
int orc_strong_remainder(const uint8_t *image, int w, int h, int c, int k, int16_t *rem) {
    if (check_dims(w, h, c, k)) return -1;
    int nbr = h / 8, nbc = w / 8;
    size_t nb = (size_t)c * nbr * nbc;
    double *coef = (double *)malloc(sizeof(double) * 64 * nb);
    int32_t *B = (int32_t *)malloc(sizeof(int32_t) * 64 * 64);
    if (!coef || !B) { free(coef); free(B); return -3; }
    orc_strong_basis(B);
    orc_dct_coefficients(image, w, h, c, coef);
    for (int ch = 0; ch < c; ch++)
        for (int br = 0; br < nbr; br++)
            for (int bc = 0; bc < nbc; bc++) {
                size_t b = ((size_t)ch * nbr + br) * nbc + bc;
                for (int p = 0; p < 64; p++) {
                    int64_t acc = 16384;
                    for (int z = 0; z <= k; z++) acc += quantise8((float)coef[64 * b + z]) * (int64_t)B[64 * z + p];
                    int64_t fl = (acc >= 0) ? (acc >> 15) : -((-acc + 32767) >> 15);
                    size_t at = ((size_t)(8 * br + p / 8) * w + (8 * bc + p % 8)) * c + ch;
                    rem[at] = (int16_t)((int64_t)image[at] - fl);
                }
            }
    free(coef); free(B);
    return 0;
}
