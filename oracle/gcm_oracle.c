/*
 * gcm_oracle.c -- plain, slow, obviously-correct CPU AES-GCM.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the parity oracle for the CUDA path in paper_2602_23067_b200/csrc/.  It shares no
 * code, header, table or constant generator with it.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It is never tuned.
 *
 * What it computes: exactly the standard AES-GCM result, written as the plain definition.
 * The paper (section 3.3.1, Eq. 1) gives only the serial GHASH recurrence
 *        Y_i = (Y_{i-1} xor X_i) . H
 * and adopts NIST SP 800-38D / FIPS-197 by reference.  Every other step
 * follows SURVEY.md section 8(c), steps 1-9, in that order and notation; the readings S1-S6 of the
 * places where the paper is silent are listed in DESIGN.md.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): installed OpenSSL (AES-ECB single block,
 * GMAC special case, whole GCM), field axioms + Frobenius a^(2^128) = a (pins the reduction
 * constant), closed forms (S(0) = 0x63, a = len = 0 => T = E_K(J0)), InvCipher(Cipher(x)) = x,
 * CTR prefix/keystream properties, GHASH linearity, segmented-GHASH = Horner by brute force,
 * tamper detection.  Nothing here is "parity unpinned".
 *
 * Style: byte-wise AES (no T-tables), bit-serial GF(2^128) multiply, sequential Horner GHASH.
 * No intrinsics, no tables beyond the S-box, which is GENERATED from its definition, not typed.
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------
 * Step 1 (FIPS-197 5.1.1): S(a) = Aff(a^-1), a^-1 the inverse in GF(2^8) modulo
 * x^8+x^4+x^3+x+1 (0 -> 0); Aff: b_i = a_i ^ a_(i+4) ^ a_(i+5) ^ a_(i+6) ^ a_(i+7) ^ c_i, c = 0x63.
 * ------------------------------------------------------------------------------------------ */
static uint8_t g_sbox[256];
static uint8_t g_inv_sbox[256];
static int g_sbox_ready = 0;

/* multiply in GF(2^8) modulo 0x11B, shift-and-add */
static uint8_t gf8_mul(uint8_t a, uint8_t b)
{
    uint8_t p = 0;
    for (int i = 0; i < 8; i++) {
        if (b & 1) p ^= a;
        uint8_t hi = a & 0x80;
        a = (uint8_t)(a << 1);
        if (hi) a ^= 0x1B;
        b >>= 1;
    }
    return p;
}

void orc_sbox_generate(uint8_t sbox[256], uint8_t inv_sbox[256])
{
    for (int a = 0; a < 256; a++) {
        /* inverse by exhaustive search: the b with a*b = 1 (0 maps to 0) */
        uint8_t inv = 0;
        if (a != 0) {
            for (int b = 1; b < 256; b++) {
                if (gf8_mul((uint8_t)a, (uint8_t)b) == 1) { inv = (uint8_t)b; break; }
            }
        }
        uint8_t out = 0;
        for (int i = 0; i < 8; i++) {
            int bit = ((inv >> i) & 1) ^ ((inv >> ((i + 4) & 7)) & 1) ^ ((inv >> ((i + 5) & 7)) & 1)
                    ^ ((inv >> ((i + 6) & 7)) & 1) ^ ((inv >> ((i + 7) & 7)) & 1) ^ ((0x63 >> i) & 1);
            out |= (uint8_t)(bit << i);
        }
        sbox[a] = out;
    }
    for (int a = 0; a < 256; a++) inv_sbox[sbox[a]] = (uint8_t)a;
}

static void sbox_init(void)
{
    if (!g_sbox_ready) {
        orc_sbox_generate(g_sbox, g_inv_sbox);
        g_sbox_ready = 1;
    }
}

/* call once from a single thread before using the oracle from several threads */
void orc_init(void) { sbox_init(); }

/* ------------------------------------------------------------------------------------------
 * Step 2 (FIPS-197 5.2): key expansion.  Nk = 4 / 8 words, Nr = 10 / 14.
 * w[i] = key words (big-endian) for i < Nk; for i >= Nk: t = w[i-1];
 *   if i mod Nk = 0: t = SubWord(RotWord(t)) ^ (x^(i/Nk - 1) in the top byte);
 *   else if Nk = 8 and i mod 8 = 4: t = SubWord(t);
 * w[i] = w[i-Nk] ^ t.
 * Returns Nr, or -1 if key_bits is not 128 or 256 (reading S1: both sizes, nothing else).
 * ------------------------------------------------------------------------------------------ */
static uint32_t sub_word(uint32_t w)
{
    return ((uint32_t)g_sbox[(w >> 24) & 0xFF] << 24) | ((uint32_t)g_sbox[(w >> 16) & 0xFF] << 16)
         | ((uint32_t)g_sbox[(w >> 8) & 0xFF] << 8) | (uint32_t)g_sbox[w & 0xFF];
}

int orc_key_expand(const uint8_t *key, int key_bits, uint32_t w[60])
{
    sbox_init();
    int Nk, Nr;
    if (key_bits == 128) { Nk = 4; Nr = 10; }
    else if (key_bits == 256) { Nk = 8; Nr = 14; }
    else return -1;
    for (int i = 0; i < Nk; i++)
        w[i] = ((uint32_t)key[4 * i] << 24) | ((uint32_t)key[4 * i + 1] << 16)
             | ((uint32_t)key[4 * i + 2] << 8) | (uint32_t)key[4 * i + 3];
    uint8_t rcon = 1; /* x^(i/Nk - 1), starts at x^0 */
    for (int i = Nk; i < 4 * (Nr + 1); i++) {
        uint32_t t = w[i - 1];
        if (i % Nk == 0) {
            t = (t << 8) | (t >> 24);                 /* RotWord */
            t = sub_word(t) ^ ((uint32_t)rcon << 24);
            rcon = gf8_mul(rcon, 2);
        } else if (Nk == 8 && i % 8 == 4) {
            t = sub_word(t);
        }
        w[i] = w[i - Nk] ^ t;
    }
    return Nr;
}

/* ------------------------------------------------------------------------------------------
 * Step 3 (FIPS-197 5.1): block encrypt.  Column-major state s[r][c] = in[r + 4c];
 * AddRoundKey(0); Nr-1 x {SubBytes, ShiftRows (row r rotates left by r), MixColumns
 * ({02,03,01,01} circulant), AddRoundKey}; final round without MixColumns.
 * ------------------------------------------------------------------------------------------ */
static void add_round_key(uint8_t s[16], const uint32_t *w, int round)
{
    for (int c = 0; c < 4; c++) {
        uint32_t k = w[4 * round + c];
        s[4 * c + 0] ^= (uint8_t)(k >> 24);
        s[4 * c + 1] ^= (uint8_t)(k >> 16);
        s[4 * c + 2] ^= (uint8_t)(k >> 8);
        s[4 * c + 3] ^= (uint8_t)k;
    }
}

static void sub_bytes(uint8_t s[16], const uint8_t box[256])
{
    for (int i = 0; i < 16; i++) s[i] = box[s[i]];
}

static void shift_rows(uint8_t s[16])
{
    uint8_t t[16];
    for (int r = 0; r < 4; r++)
        for (int c = 0; c < 4; c++)
            t[r + 4 * c] = s[r + 4 * ((c + r) & 3)];
    memcpy(s, t, 16);
}

static void inv_shift_rows(uint8_t s[16])
{
    uint8_t t[16];
    for (int r = 0; r < 4; r++)
        for (int c = 0; c < 4; c++)
            t[r + 4 * ((c + r) & 3)] = s[r + 4 * c];
    memcpy(s, t, 16);
}

/* FIPS-197 4.2.1: xtime(a) = a . {02}: shift left, xor 0x1B if the dropped bit was set */
static uint8_t xtime(uint8_t a)
{
    return (uint8_t)((a << 1) ^ ((a & 0x80) ? 0x1B : 0x00));
}

static void mix_columns(uint8_t s[16])
{
    for (int c = 0; c < 4; c++) {
        uint8_t a0 = s[4 * c], a1 = s[4 * c + 1], a2 = s[4 * c + 2], a3 = s[4 * c + 3];
        /* {02}.a = xtime(a); {03}.a = xtime(a) ^ a */
        s[4 * c + 0] = (uint8_t)(xtime(a0) ^ (xtime(a1) ^ a1) ^ a2 ^ a3);
        s[4 * c + 1] = (uint8_t)(a0 ^ xtime(a1) ^ (xtime(a2) ^ a2) ^ a3);
        s[4 * c + 2] = (uint8_t)(a0 ^ a1 ^ xtime(a2) ^ (xtime(a3) ^ a3));
        s[4 * c + 3] = (uint8_t)((xtime(a0) ^ a0) ^ a1 ^ a2 ^ xtime(a3));
    }
}

static void inv_mix_columns(uint8_t s[16])
{
    for (int c = 0; c < 4; c++) {
        uint8_t a0 = s[4 * c], a1 = s[4 * c + 1], a2 = s[4 * c + 2], a3 = s[4 * c + 3];
        s[4 * c + 0] = gf8_mul(a0, 14) ^ gf8_mul(a1, 11) ^ gf8_mul(a2, 13) ^ gf8_mul(a3, 9);
        s[4 * c + 1] = gf8_mul(a0, 9) ^ gf8_mul(a1, 14) ^ gf8_mul(a2, 11) ^ gf8_mul(a3, 13);
        s[4 * c + 2] = gf8_mul(a0, 13) ^ gf8_mul(a1, 9) ^ gf8_mul(a2, 14) ^ gf8_mul(a3, 11);
        s[4 * c + 3] = gf8_mul(a0, 11) ^ gf8_mul(a1, 13) ^ gf8_mul(a2, 9) ^ gf8_mul(a3, 14);
    }
}

void orc_encrypt_block(const uint32_t *w, int Nr, const uint8_t in[16], uint8_t out[16])
{
    uint8_t s[16];
    memcpy(s, in, 16);
    add_round_key(s, w, 0);
    for (int round = 1; round < Nr; round++) {
        sub_bytes(s, g_sbox);
        shift_rows(s);
        mix_columns(s);
        add_round_key(s, w, round);
    }
    sub_bytes(s, g_sbox);
    shift_rows(s);
    add_round_key(s, w, Nr);
    memcpy(out, s, 16);
}

/* FIPS-197 5.3 inverse cipher; used only by the pin InvCipher(Cipher(x)) = x, never by GCM */
void orc_decrypt_block(const uint32_t *w, int Nr, const uint8_t in[16], uint8_t out[16])
{
    uint8_t s[16];
    memcpy(s, in, 16);
    add_round_key(s, w, Nr);
    for (int round = Nr - 1; round >= 1; round--) {
        inv_shift_rows(s);
        sub_bytes(s, g_inv_sbox);
        add_round_key(s, w, round);
        inv_mix_columns(s);
    }
    inv_shift_rows(s);
    sub_bytes(s, g_inv_sbox);
    add_round_key(s, w, 0);
    memcpy(out, s, 16);
}

/* ------------------------------------------------------------------------------------------
 * Step 6 (SP 800-38D Algorithm 1): Z = X . Y in GF(2^128).
 * Bit i of a block = bit (7 - i mod 8) of byte floor(i/8), i.e. byte 0's most significant bit is
 * the coefficient of x^0.  Z = 0, V = Y; for i = 0..127: if x_i: Z ^= V;
 * V = (V >> 1) ^ (lsb(V) ? R : 0), R = 0xE1 || 0^120; ">>" acts on the 128-bit string with byte 0
 * leftmost.  The 128-bit string is held as two big-endian 64-bit halves (hi = bytes 0..7).
 * ------------------------------------------------------------------------------------------ */
typedef struct { uint64_t hi, lo; } blk128;

static blk128 load_be(const uint8_t b[16])
{
    blk128 v = {0, 0};
    for (int i = 0; i < 8; i++) v.hi = (v.hi << 8) | b[i];
    for (int i = 8; i < 16; i++) v.lo = (v.lo << 8) | b[i];
    return v;
}

static void store_be(blk128 v, uint8_t b[16])
{
    for (int i = 7; i >= 0; i--) { b[i] = (uint8_t)v.hi; v.hi >>= 8; }
    for (int i = 15; i >= 8; i--) { b[i] = (uint8_t)v.lo; v.lo >>= 8; }
}

static blk128 gf128_mul(blk128 X, blk128 Y)
{
    blk128 Z = {0, 0};
    blk128 V = Y;
    for (int i = 0; i < 128; i++) {
        uint64_t xi = (i < 64) ? (X.hi >> (63 - i)) & 1 : (X.lo >> (127 - i)) & 1;
        if (xi) { Z.hi ^= V.hi; Z.lo ^= V.lo; }
        uint64_t lsb = V.lo & 1;
        V.lo = (V.lo >> 1) | (V.hi << 63);
        V.hi = V.hi >> 1;
        if (lsb) V.hi ^= 0xE100000000000000ULL;
    }
    return Z;
}

void orc_gf_mul(const uint8_t X[16], const uint8_t Y[16], uint8_t Z[16])
{
    store_be(gf128_mul(load_be(X), load_be(Y)), Z);
}

/* H^e by repeated multiplication, square-and-multiply over the bits of e (e = 0 gives the field's
 * one, 0x80 || 0^120).  Used by the segmented-GHASH identity below and by tests. */
void orc_gf_pow(const uint8_t H[16], uint64_t e, uint8_t out[16])
{
    blk128 result = {0x8000000000000000ULL, 0};
    blk128 base = load_be(H);
    while (e) {
        if (e & 1) result = gf128_mul(result, base);
        base = gf128_mul(base, base);
        e >>= 1;
    }
    store_be(result, out);
}

/* ------------------------------------------------------------------------------------------
 * Step 7 (Eq. 1): GHASH, the serial recurrence.
 * orc_ghash_update continues Y over the 16-byte blocks of `data`, the last one zero-padded
 * (reading S4: A and C are padded separately, so call it once for A and once for C).
 * ------------------------------------------------------------------------------------------ */
void orc_ghash_update(const uint8_t H[16], uint8_t Y[16], const uint8_t *data, uint64_t len)
{
    blk128 h = load_be(H);
    blk128 y = load_be(Y);
    uint64_t off = 0;
    while (off < len) {
        uint8_t x[16] = {0};
        uint64_t take = (len - off < 16) ? (len - off) : 16;
        memcpy(x, data + off, (size_t)take);
        blk128 xb = load_be(x);
        y.hi ^= xb.hi; y.lo ^= xb.lo;            /* Y_{i-1} xor X_i */
        y = gf128_mul(y, h);                      /* . H             */
        off += take;
    }
    store_be(y, Y);
}

static void length_block(uint64_t aad_len, uint64_t len, uint8_t L[16])
{
    uint64_t abits = aad_len * 8, cbits = len * 8;   /* reading S3: BE64(bits of A) || BE64(bits of C) */
    for (int i = 7; i >= 0; i--) { L[i] = (uint8_t)abits; abits >>= 8; }
    for (int i = 15; i >= 8; i--) { L[i] = (uint8_t)cbits; cbits >>= 8; }
}

/* S = GHASH_H(A || 0-pad || C || 0-pad || len64(A) || len64(C)) */
void orc_ghash(const uint8_t H[16], const uint8_t *aad, uint64_t aad_len,
               const uint8_t *c, uint64_t len, uint8_t S[16])
{
    uint8_t L[16];
    memset(S, 0, 16);
    orc_ghash_update(H, S, aad, aad_len);
    orc_ghash_update(H, S, c, len);
    length_block(aad_len, len, L);
    orc_ghash_update(H, S, L, 16);
}

/* ------------------------------------------------------------------------------------------
 * Segmented GHASH -- NOT the definition; an identity derived from it, kept here so that a 4 GiB
 * tag can be checked in under a minute on several host threads:
 *   Horner over blocks X_1..X_N equals  XOR_k  Horner(segment k) . H^(number of blocks after it).
 * orc_ghash_segment returns Horner(segment) . H^blocks_after for one run of whole blocks (the
 * last block may be partial and is zero-padded).  tests/test_oracle_ghash.py pins this against
 * orc_ghash by brute force for every N up to several hundred and every split point; callers
 * XOR the segment values (the Python side in oracle.py does, optionally on threads).
 * ------------------------------------------------------------------------------------------ */
void orc_ghash_segment(const uint8_t H[16], const uint8_t *data, uint64_t len,
                       uint64_t blocks_after, uint8_t out[16])
{
    uint8_t y[16] = {0}, p[16];
    orc_ghash_update(H, y, data, len);
    orc_gf_pow(H, blocks_after, p);
    orc_gf_mul(y, p, out);
}

/* ------------------------------------------------------------------------------------------
 * Steps 4-5: H = E_K(0^128); J0 = IV || 00 00 00 01;
 * CTR: for g = 0..n-1: KS = E_K(IV || BE32(g + 2)); C[16g..] = P[16g..] ^ KS, truncated at len
 * (reading S2: payload block g uses counter value g + 2; the counter depends
 * on the block index only).  `first_block` lets callers process a byte range that starts at
 * block index first_block (must be the start of a block); that is how several host threads share
 * one message in the cpu_baseline leg.
 * ------------------------------------------------------------------------------------------ */
void orc_ctr_xor_w(const uint32_t *w, int Nr, const uint8_t iv[12], uint64_t first_block,
                   const uint8_t *in, uint8_t *out, uint64_t len)
{
    uint8_t ctr[16], ks[16];
    memcpy(ctr, iv, 12);
    uint64_t off = 0, g = first_block;
    while (off < len) {
        uint32_t c32 = (uint32_t)(g + 2);
        ctr[12] = (uint8_t)(c32 >> 24); ctr[13] = (uint8_t)(c32 >> 16);
        ctr[14] = (uint8_t)(c32 >> 8);  ctr[15] = (uint8_t)c32;
        orc_encrypt_block(w, Nr, ctr, ks);
        uint64_t take = (len - off < 16) ? (len - off) : 16;
        for (uint64_t i = 0; i < take; i++) out[off + i] = in[off + i] ^ ks[i];
        off += take;
        g++;
    }
}

int orc_ctr_xor(const uint8_t *key, int key_bits, const uint8_t iv[12], uint64_t first_block,
                const uint8_t *in, uint8_t *out, uint64_t len)
{
    uint32_t w[60];
    int Nr = orc_key_expand(key, key_bits, w);
    if (Nr < 0) return -1;
    orc_ctr_xor_w(w, Nr, iv, first_block, in, out, len);
    return 0;
}

/* H = E_K(0^128) and E_K(J0), J0 = IV || 0^31 || 1 */
int orc_hash_subkey(const uint8_t *key, int key_bits, uint8_t H[16])
{
    uint32_t w[60];
    uint8_t zero[16] = {0};
    int Nr = orc_key_expand(key, key_bits, w);
    if (Nr < 0) return -1;
    orc_encrypt_block(w, Nr, zero, H);
    return 0;
}

int orc_ek_j0(const uint8_t *key, int key_bits, const uint8_t iv[12], uint8_t out[16])
{
    uint32_t w[60];
    uint8_t j0[16];
    int Nr = orc_key_expand(key, key_bits, w);
    if (Nr < 0) return -1;
    memcpy(j0, iv, 12);
    j0[12] = 0; j0[13] = 0; j0[14] = 0; j0[15] = 1;
    orc_encrypt_block(w, Nr, j0, out);
    return 0;
}

/* single-block ECB, for the OpenSSL pin of steps 1-3 */
int orc_ecb_block(const uint8_t *key, int key_bits, const uint8_t in[16], uint8_t out[16], int decrypt)
{
    uint32_t w[60];
    int Nr = orc_key_expand(key, key_bits, w);
    if (Nr < 0) return -1;
    if (decrypt) orc_decrypt_block(w, Nr, in, out);
    else orc_encrypt_block(w, Nr, in, out);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Step 8: T = E_K(J0) ^ GHASH.   Whole-function entry points.
 * Limits (SP 800-38D): len <= 2^36 - 32 bytes.  Returns 0, or -1 bad key size, -2 bad length.
 * ------------------------------------------------------------------------------------------ */
int orc_gcm_encrypt(const uint8_t *key, int key_bits, const uint8_t iv[12],
                    const uint8_t *aad, uint64_t aad_len,
                    const uint8_t *pt, uint64_t len, uint8_t *ct, uint8_t tag[16])
{
    uint8_t H[16], S[16], EJ0[16];
    if (len > ((1ULL << 36) - 32)) return -2;
    if (orc_hash_subkey(key, key_bits, H) < 0) return -1;
    orc_ctr_xor(key, key_bits, iv, 0, pt, ct, len);
    orc_ghash(H, aad, aad_len, ct, len, S);
    orc_ek_j0(key, key_bits, iv, EJ0);
    for (int i = 0; i < 16; i++) tag[i] = EJ0[i] ^ S[i];
    return 0;
}

/* Step 9: recompute T' from (IV, A, C); diff = OR of all 16 byte-XORs (no early
 * exit); if diff != 0 -> authentication failure, output all zeros (payload
 * suppression by memset; L219: validation gate); else P = C ^ KS.  Returns 0 ok, 1 auth failure,
 * <0 argument error. */
int orc_gcm_decrypt_verify(const uint8_t *key, int key_bits, const uint8_t iv[12],
                           const uint8_t *aad, uint64_t aad_len,
                           const uint8_t *ct, uint64_t len, uint8_t *pt, const uint8_t tag[16])
{
    uint8_t H[16], S[16], EJ0[16];
    if (len > ((1ULL << 36) - 32)) return -2;
    if (orc_hash_subkey(key, key_bits, H) < 0) return -1;
    orc_ghash(H, aad, aad_len, ct, len, S);
    orc_ek_j0(key, key_bits, iv, EJ0);
    uint8_t diff = 0;
    for (int i = 0; i < 16; i++) diff |= (uint8_t)(EJ0[i] ^ S[i] ^ tag[i]);
    if (diff != 0) {
        memset(pt, 0, (size_t)len);
        return 1;
    }
    orc_ctr_xor(key, key_bits, iv, 0, ct, pt, len);
    return 0;
}
