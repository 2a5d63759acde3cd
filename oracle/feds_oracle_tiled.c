/*
 * feds_oracle_tiled.c — CPU ORACLE for the report's own DWT design: selective encryption of 8x8 tiles with two levels of the
 * integer Le Gall 5/3 transform, AES on the "level 1" coefficients and SHA-256 / SHA-512 keystreams on levels 2 and 3 (PAPER.md
 * 6.9.3-6.9.4, Figure 18). TEST INFRASTRUCTURE, NOT PRODUCT (see feds_oracle.c).
 *
 * What the report says: every 8x8 block gets two successive DWT levels; the low-frequency k = 4 coefficients ("level 1") are
 * protected by AES-128; they "generate a bit sequence with a length of 256" by SHA-256, "also with the AES key and IV", that is
 * XORed over the rest of the second-level coefficients ("level 2"); level 2 generates 512 bits by SHA-512, also with key and IV,
 * XORed over the first-level subbands ("level 3"). Storage: 10 bits per first-level coefficient; second
 * level "11-bits for each of the [...] four coefficients [of one corner] and 10-bits for rest"; 40 + 124 = 164 bits confidential,
 * 480 bits public, 644 in all. DESIGN.md section 2.5 fixes what is left open (readings T1-T8):
 *   T1  per channel plane, per 8x8 tile: x - 128 (A13), 5/3 lifting of DESIGN.md 2.2 on the tile (rows then columns, whole-sample
 *       symmetric extension at the TILE borders), then again on its 4x4 LL.
 *   T2  level 1 = LL2 (4 values, row-major); level 2 = HL2, LH2, HH2 (4 each, row-major); level 3 = HL1, LH1, HH1 (16 each).
 *   T3  fields are two's complement, 10 bits, except HH2: 11 bits (the only subband whose range, +-648, needs them; the linear
 *       bounds are LL2 338, HL2/LH2 468, HL1/LH1 384, HH1 511 -- tests search the extremes); each level is one little-endian bit
 *       stream (fields LSB first) padded with zero bits to whole bytes: 5, 16 (124 bits) and 60 bytes.
 *   T4  K2 = SHA-256(level-1 bytes || key || IV), K3 = SHA-512(level-2 bytes || key || IV), plaintext bytes as packed (pad bits zero),
 *       IV = the image's 16-byte nonce; stored level 2 = its 16 bytes XOR K2[0..15], stored level 3 = its 60 bytes XOR K3[0..59].
 *   T5  private fragment = [stored level-2 bytes, 16 per tile] || [level-1 bytes of all tiles, 5 per tile, as ONE AES-128-CTR message];
 *       public fragment = stored level-3 bytes, 60 per tile. Tile order: channel, tile row, tile column. 21 private bytes per 64
 *       pixels = 32.8 % ("at most 32%"), 81 bytes in all = 126.6 % ("about 26% more"; 4 pad bits per tile more than 644 bits).
 *   T6  digests: the stream Merkle layout of DESIGN.md 2.2 (2048-byte leaves, fan-out 16) over each fragment as stored.
 *   T7  inverse: AES-decrypt level 1, K2 -> level 2, K3 -> level 3, unpack, inverse transform, + 128, clamp to a byte.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* from the other oracle files */
void orc_sha256(const uint8_t *msg, uint64_t n, uint8_t out[32]);
void orc_sha512(const uint8_t *msg, uint64_t n, uint8_t out[64]);
void orc_dwt53_fwd_1d(const int32_t *x, int N, int32_t *y);
void orc_dwt53_inv_1d(const int32_t *y, int N, int32_t *x);
void orc_aes128_ctr_xor(const uint8_t key[16], const uint8_t nonce[16], uint64_t first_block, uint8_t *buf, uint64_t n);
int orc_merkle_stream(const uint8_t *bytes, uint64_t n, uint64_t leaf_bytes, int F, uint8_t root[32]);

static int check_dims(int w, int h, int c) {
    if (w <= 0 || h <= 0 || (w % 8) || (h % 8)) return -1;
    if (!(c == 1 || c == 3 || c == 4)) return -2;
    return 0;
}

/* one 2-D level on the top-left n x n corner of an 8x8 row-major tile: rows, then columns (T1) */
static void level_fwd(int32_t t[64], int n) {
    int32_t in[8], out[8];
    for (int r = 0; r < n; r++) {
        for (int i = 0; i < n; i++) in[i] = t[8 * r + i];
        orc_dwt53_fwd_1d(in, n, out);
        for (int i = 0; i < n; i++) t[8 * r + i] = out[i];
    }
    for (int c = 0; c < n; c++) {
        for (int i = 0; i < n; i++) in[i] = t[8 * i + c];
        orc_dwt53_fwd_1d(in, n, out);
        for (int i = 0; i < n; i++) t[8 * i + c] = out[i];
    }
}
static void level_inv(int32_t t[64], int n) {
    int32_t in[8], out[8];
    for (int c = 0; c < n; c++) {
        for (int i = 0; i < n; i++) in[i] = t[8 * i + c];
        orc_dwt53_inv_1d(in, n, out);
        for (int i = 0; i < n; i++) t[8 * i + c] = out[i];
    }
    for (int r = 0; r < n; r++) {
        for (int i = 0; i < n; i++) in[i] = t[8 * r + i];
        orc_dwt53_inv_1d(in, n, out);
        for (int i = 0; i < n; i++) t[8 * r + i] = out[i];
    }
}

/* the 64 coefficients of a tile in level order (T2): [0,4) LL2, [4,8) HL2, [8,12) LH2, [12,16) HH2, [16,32) HL1, [32,48) LH1, [48,64) HH1 */
void orc_tiled_forward(const uint8_t pixels[64], int32_t coef[64]) {
    int32_t t[64];
    for (int i = 0; i < 64; i++) t[i] = (int32_t)pixels[i] - 128;
    level_fwd(t, 8);
    level_fwd(t, 4);
    int n = 0;
    for (int r = 0; r < 2; r++) for (int c = 0; c < 2; c++) coef[n++] = t[8 * r + c];           /* LL2 */
    for (int r = 0; r < 2; r++) for (int c = 2; c < 4; c++) coef[n++] = t[8 * r + c];           /* HL2: high-pass horizontally */
    for (int r = 2; r < 4; r++) for (int c = 0; c < 2; c++) coef[n++] = t[8 * r + c];           /* LH2 */
    for (int r = 2; r < 4; r++) for (int c = 2; c < 4; c++) coef[n++] = t[8 * r + c];           /* HH2 */
    for (int r = 0; r < 4; r++) for (int c = 4; c < 8; c++) coef[n++] = t[8 * r + c];           /* HL1 */
    for (int r = 4; r < 8; r++) for (int c = 0; c < 4; c++) coef[n++] = t[8 * r + c];           /* LH1 */
    for (int r = 4; r < 8; r++) for (int c = 4; c < 8; c++) coef[n++] = t[8 * r + c];           /* HH1 */
}
void orc_tiled_inverse(const int32_t coef[64], uint8_t pixels[64]) {
    int32_t t[64];
    int n = 0;
    for (int r = 0; r < 2; r++) for (int c = 0; c < 2; c++) t[8 * r + c] = coef[n++];
    for (int r = 0; r < 2; r++) for (int c = 2; c < 4; c++) t[8 * r + c] = coef[n++];
    for (int r = 2; r < 4; r++) for (int c = 0; c < 2; c++) t[8 * r + c] = coef[n++];
    for (int r = 2; r < 4; r++) for (int c = 2; c < 4; c++) t[8 * r + c] = coef[n++];
    for (int r = 0; r < 4; r++) for (int c = 4; c < 8; c++) t[8 * r + c] = coef[n++];
    for (int r = 4; r < 8; r++) for (int c = 0; c < 4; c++) t[8 * r + c] = coef[n++];
    for (int r = 4; r < 8; r++) for (int c = 4; c < 8; c++) t[8 * r + c] = coef[n++];
    level_inv(t, 4);
    level_inv(t, 8);
    for (int i = 0; i < 64; i++) {
        int32_t v = t[i] + 128;
        pixels[i] = (uint8_t)(v < 0 ? 0 : (v > 255 ? 255 : v));
    }
}

static int field_bits(int i) { return (i >= 12 && i < 16) ? 11 : 10; } /* T3: HH2 takes 11 bits */

/* T3: coefficients [lo, hi) -> little-endian bit stream of two's complement fields; returns 0, or -1 if a value does not fit */
static int pack_level(const int32_t *coef, int lo, int hi, uint8_t *out, int nbytes) {
    memset(out, 0, (size_t)nbytes);
    int pos = 0;
    for (int i = lo; i < hi; i++) {
        int b = field_bits(i);
        if (coef[i] < -(1 << (b - 1)) || coef[i] > (1 << (b - 1)) - 1) return -1;
        uint32_t f = (uint32_t)coef[i] & ((1u << b) - 1u);
        for (int k = 0; k < b; k++, pos++)
            if ((f >> k) & 1u) out[pos / 8] |= (uint8_t)(1u << (pos % 8));
    }
    return 0;
}
static void unpack_level(const uint8_t *in, int lo, int hi, int32_t *coef) {
    int pos = 0;
    for (int i = lo; i < hi; i++) {
        int b = field_bits(i);
        uint32_t f = 0;
        for (int k = 0; k < b; k++, pos++)
            if ((in[pos / 8] >> (pos % 8)) & 1u) f |= 1u << k;
        coef[i] = (f & (1u << (b - 1))) ? (int32_t)f - (1 << b) : (int32_t)f;
    }
}

/* packed plaintext levels of one tile: l1[5], l2[16], l3[60] */
int orc_tiled_pack(const int32_t coef[64], uint8_t l1[5], uint8_t l2[16], uint8_t l3[60]) {
    if (pack_level(coef, 0, 4, l1, 5)) return -1;
    if (pack_level(coef, 4, 16, l2, 16)) return -1;
    return pack_level(coef, 16, 64, l3, 60);
}

uint64_t orc_tiled_private_bytes(int w, int h, int c) { return check_dims(w, h, c) ? 0 : (uint64_t)(w / 8) * (h / 8) * c * 21; }
uint64_t orc_tiled_public_bytes(int w, int h, int c) { return check_dims(w, h, c) ? 0 : (uint64_t)(w / 8) * (h / 8) * c * 60; }

static void keystreams(const uint8_t l1[5], const uint8_t l2[16], const uint8_t key[16], const uint8_t iv[16], uint8_t k2[32], uint8_t k3[64]) {
    uint8_t m[48];
    if (k2) { memcpy(m, l1, 5); memcpy(m + 5, key, 16); memcpy(m + 21, iv, 16); orc_sha256(m, 37, k2); }   /* T4 */
    if (k3) { memcpy(m, l2, 16); memcpy(m + 16, key, 16); memcpy(m + 32, iv, 16); orc_sha512(m, 48, k3); }
}

int orc_fragment_tiled(const uint8_t *image, int w, int h, int c, const uint8_t key[16], const uint8_t nonce[16], uint64_t leaf_bytes,
                       int F, uint8_t *priv, uint8_t *pub, uint8_t digests[64]) {
    if (check_dims(w, h, c)) return -1;
    int ntr = h / 8, ntc = w / 8;
    uint64_t T = (uint64_t)c * ntr * ntc;
    uint8_t *secB = priv, *secA = priv + 16 * T;   /* T5 */
    for (int ch = 0; ch < c; ch++)
        for (int tr = 0; tr < ntr; tr++)
            for (int tc = 0; tc < ntc; tc++) {
                uint64_t t = ((uint64_t)ch * ntr + tr) * ntc + tc;
                uint8_t px[64], l1[5], l2[16], l3[60], k2[32], k3[64];
                int32_t coef[64];
                for (int i = 0; i < 8; i++)
                    for (int j = 0; j < 8; j++) px[8 * i + j] = image[((size_t)(8 * tr + i) * w + (8 * tc + j)) * c + ch];
                orc_tiled_forward(px, coef);
                if (orc_tiled_pack(coef, l1, l2, l3)) return -4;
                keystreams(l1, l2, key, nonce, k2, k3);
                memcpy(secA + 5 * t, l1, 5);
                for (int i = 0; i < 16; i++) secB[16 * t + i] = (uint8_t)(l2[i] ^ k2[i]);
                for (int i = 0; i < 60; i++) pub[60 * t + i] = (uint8_t)(l3[i] ^ k3[i]);
            }
    orc_aes128_ctr_xor(key, nonce, 0, secA, 5 * T);   /* T5: the level-1 section is one CTR message */
    int rc = orc_merkle_stream(priv, 21 * T, leaf_bytes, F, digests);
    if (rc) return rc;
    return orc_merkle_stream(pub, 60 * T, leaf_bytes, F, digests + 32);
}

int orc_defragment_tiled(const uint8_t *priv, const uint8_t *pub, int w, int h, int c, const uint8_t key[16], const uint8_t nonce[16],
                         uint64_t leaf_bytes, int F, const uint8_t *expected, uint8_t *image_out, uint32_t *flags) {
    if (check_dims(w, h, c)) return -1;
    int ntr = h / 8, ntc = w / 8;
    uint64_t T = (uint64_t)c * ntr * ntc;
    if (flags) *flags = 0;
    if (expected) {
        uint8_t dg[64];
        orc_merkle_stream(priv, 21 * T, leaf_bytes, F, dg);
        orc_merkle_stream(pub, 60 * T, leaf_bytes, F, dg + 32);
        uint32_t fl = 0;
        if (memcmp(dg, expected, 32)) fl |= 1u;
        if (memcmp(dg + 32, expected + 32, 32)) fl |= 2u;
        if (flags) *flags = fl;
    }
    uint8_t *secA = (uint8_t *)malloc(T ? 5 * T : 1);
    if (!secA) return -3;
    memcpy(secA, priv + 16 * T, 5 * T);
    orc_aes128_ctr_xor(key, nonce, 0, secA, 5 * T);
    const uint8_t *secB = priv;
    for (int ch = 0; ch < c; ch++)
        for (int tr = 0; tr < ntr; tr++)
            for (int tc = 0; tc < ntc; tc++) {
                uint64_t t = ((uint64_t)ch * ntr + tr) * ntc + tc;
                uint8_t l2[16], l3[60], k2[32], k3[64], px[64];
                int32_t coef[64];
                keystreams(secA + 5 * t, NULL, key, nonce, k2, NULL);
                for (int i = 0; i < 16; i++) l2[i] = (uint8_t)(secB[16 * t + i] ^ k2[i]);
                l2[15] &= 0x0f;   /* the four pad bits of the 124-bit stream are zero in the plaintext (T3) and enter K3 as zeros */
                keystreams(NULL, l2, key, nonce, NULL, k3);
                for (int i = 0; i < 60; i++) l3[i] = (uint8_t)(pub[60 * t + i] ^ k3[i]);
                unpack_level(secA + 5 * t, 0, 4, coef);
                unpack_level(l2, 4, 16, coef);
                unpack_level(l3, 16, 64, coef);
                orc_tiled_inverse(coef, px);
                for (int i = 0; i < 8; i++)
                    for (int j = 0; j < 8; j++) image_out[((size_t)(8 * tr + i) * w + (8 * tc + j)) * c + ch] = px[8 * i + j];
            }
    free(secA);
    return 0;
}
