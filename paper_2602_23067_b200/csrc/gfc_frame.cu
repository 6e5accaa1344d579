// gfc_frame.cu -- the authenticated FITS container (include/gfc.h): PAPER.md section 3.2.2-3.2.3
// (L113-L157), the dual-stream pipeline of section 3.3.2 (L209-L219) and the access scenarios of
// section 4.2 (L237-L245, Table 2).
//
// Host side: 80-character card parsing / formatting, hex text, the CHECKSUM character encoding and
// stream orchestration.  Everything cryptographic (key schedule, H powers, CTR, GHASH, tag, compare)
// and the DATASUM of the payload run in the CUDA kernels of this library; nothing here falls back to
// the CPU.  Shares nothing with oracle/.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <string>
#include <vector>

#include "../../include/gfc.h"
#include "gcm_common.cuh"
#include "gcm_api_internal.h"
#include "fits_sum.cuh"

namespace {

constexpr uint64_t kBlock = 2880;
constexpr uint64_t kCard = 80;

// ---- cards (FITS standard 4.0 section 4.2, fixed format) ------------------------------------------
void put_card(std::string &h, const std::string &text)
{
    std::string c = text.substr(0, kCard);
    c.resize(kCard, ' ');
    h += c;
}
void put_logical(std::string &h, const char *key, bool v)
{
    char b[96];
    snprintf(b, sizeof b, "%-8s= %20s", key, v ? "T" : "F");
    put_card(h, b);
}
void put_int(std::string &h, const char *key, long long v)
{
    char b[96];
    snprintf(b, sizeof b, "%-8s= %20lld", key, v);
    put_card(h, b);
}
void put_str(std::string &h, const char *key, const std::string &s)
{
    std::string v = s;
    if (v.size() < 8) v.resize(8, ' ');
    char k[16];
    snprintf(k, sizeof k, "%-8s= ", key);
    put_card(h, std::string(k) + "'" + v + "'");
}
// OGIP long-string convention: 67 characters + '&' per card, the rest on CONTINUE cards (reading F4)
void put_long_str(std::string &h, const char *key, const std::string &s)
{
    size_t pos = 0;
    bool first = true;
    do {
        std::string piece = s.substr(pos, 67);
        pos += piece.size();
        if (pos < s.size()) piece += '&';
        if (first) put_str(h, key, piece);
        else put_card(h, "CONTINUE  '" + piece + "'");
        first = false;
    } while (pos < s.size());
}
void put_end_and_pad(std::string &h)
{
    put_card(h, "END");
    h.resize((h.size() + kBlock - 1) / kBlock * kBlock, ' ');
}

// A parsed header: the cards before END and the header's length in the file (a multiple of 2880).
struct Header {
    std::vector<const char *> cards;
    uint64_t length = 0;
};

bool parse_header(const uint8_t *buf, uint64_t len, uint64_t off, Header *out)
{
    out->cards.clear();
    uint64_t pos = off;
    for (;;) {
        if (pos + kCard > len) return false;
        const char *c = (const char *)buf + pos;
        pos += kCard;
        if (memcmp(c, "END     ", 8) == 0) {
            bool blank = true;
            for (int i = 8; i < 80; i++) blank = blank && c[i] == ' ';
            if (blank) break;
        }
        out->cards.push_back(c);
    }
    out->length = (pos - off + kBlock - 1) / kBlock * kBlock;
    return off + out->length <= len;
}

const char *find_card(const Header &h, const char *key, size_t *index = nullptr)
{
    char k[16];
    snprintf(k, sizeof k, "%-8s= ", key);
    for (size_t i = 0; i < h.cards.size(); i++)
        if (memcmp(h.cards[i], k, 10) == 0) {
            if (index) *index = i;
            return h.cards[i];
        }
    return nullptr;
}

bool get_int(const Header &h, const char *key, long long *v)
{
    const char *c = find_card(h, key);
    if (!c) return false;
    char b[72];
    memcpy(b, c + 10, 70);
    b[70] = 0;
    if (char *slash = strchr(b, '/')) *slash = 0;
    char *end = nullptr;
    long long x = strtoll(b, &end, 10);
    if (end == b) return false;
    while (*end == ' ') end++;
    if (*end) return false;
    *v = x;
    return true;
}

bool quoted(const char *field, size_t n, std::string *s)      // text between the first two quotes
{
    const char *a = (const char *)memchr(field, '\'', n);
    if (!a) return false;
    const char *b = (const char *)memchr(a + 1, '\'', n - (a + 1 - field));
    if (!b) return false;
    s->assign(a + 1, b);
    while (!s->empty() && s->back() == ' ') s->pop_back();
    return true;
}

bool get_str(const Header &h, const char *key, std::string *s)   // joins CONTINUE cards
{
    size_t i = 0;
    const char *c = find_card(h, key, &i);
    if (!c || !quoted(c + 10, 70, s)) return false;
    for (size_t j = i + 1; !s->empty() && s->back() == '&' && j < h.cards.size(); j++) {
        if (memcmp(h.cards[j], "CONTINUE  ", 10) != 0) break;
        std::string more;
        if (!quoted(h.cards[j] + 10, 70, &more)) return false;
        s->pop_back();
        *s += more;
    }
    return true;
}

// ---- hex text -----------------------------------------------------------------------------------
std::string to_hex(const uint8_t *p, size_t n)
{
    static const char d[] = "0123456789ABCDEF";
    std::string s(2 * n, '0');
    for (size_t i = 0; i < n; i++) {
        s[2 * i] = d[p[i] >> 4];
        s[2 * i + 1] = d[p[i] & 15];
    }
    return s;
}
int nibble(char c)
{
    if (c >= '0' && c <= '9') return c - '0';
    if (c >= 'A' && c <= 'F') return c - 'A' + 10;
    if (c >= 'a' && c <= 'f') return c - 'a' + 10;
    return -1;
}
bool from_hex(const std::string &s, uint8_t *out, size_t n)
{
    if (s.size() != 2 * n) return false;
    for (size_t i = 0; i < n; i++) {
        int a = nibble(s[2 * i]), b = nibble(s[2 * i + 1]);
        if (a < 0 || b < 0) return false;
        out[i] = (uint8_t)(a << 4 | b);
    }
    return true;
}

// ---- FITS checksum of the (small) header text on the host; the payload's DATASUM is a kernel ------
uint32_t header_sum32(const std::string &h, uint32_t start)
{
    uint64_t s = start;
    for (size_t i = 0; i + 4 <= h.size(); i += 4)
        s += (uint32_t)(uint8_t)h[i] << 24 | (uint32_t)(uint8_t)h[i + 1] << 16 | (uint32_t)(uint8_t)h[i + 2] << 8 |
             (uint32_t)(uint8_t)h[i + 3];
    while (s >> 32) s = (s & 0xFFFFFFFFull) + (s >> 32);
    return (uint32_t)s;
}
// FITS standard 4.0 appendix J.2: 32-bit value -> 16 alphanumeric characters, rotated right by one
void checksum_chars(uint32_t value, char out[17])
{
    char asc[16];
    for (int i = 0; i < 4; i++) {
        const int byte = (value >> (24 - 8 * i)) & 0xFF;
        int ch[4] = {byte / 4 + byte % 4 + '0', byte / 4 + '0', byte / 4 + '0', byte / 4 + '0'};
        for (bool again = true; again;) {
            again = false;
            for (int j = 0; j < 4; j += 2) {
                auto punct = [](int c) { return (c >= 0x3A && c <= 0x40) || (c >= 0x5B && c <= 0x60); };
                if (punct(ch[j]) || punct(ch[j + 1])) {
                    ch[j]++;
                    ch[j + 1]--;
                    again = true;
                }
            }
        }
        for (int j = 0; j < 4; j++) asc[4 * j + i] = (char)ch[j];
    }
    for (int i = 0; i < 16; i++) out[i] = asc[(i + 15) % 16];
    out[16] = 0;
}
// appends DATASUM, CHECKSUM, END and the blank padding; sets CHECKSUM so that the HDU sums to -0
void finish_header(std::string &h, uint32_t datasum)
{
    put_str(h, "DATASUM", std::to_string(datasum));
    const size_t at = h.size();
    put_str(h, "CHECKSUM", "0000000000000000");
    put_end_and_pad(h);
    const uint32_t total = header_sum32(h, datasum);
    char enc[17];
    checksum_chars(~total, enc);
    memcpy(&h[at + 11], enc, 16);
}

}  // namespace

// ---- context ------------------------------------------------------------------------------------------
struct gfc_context {
    int device;
    int sm_count;
    uint64_t max_header, max_data;
    cudaStream_t streamH, streamD;          // header stream and data stream
    cudaEvent_t evH0, evH1, evD0, evD1;
    uint8_t *h_out;                         // pinned result buffer (L170-L171, L289)
    uint64_t out_cap;
    uint8_t *h_hdr;                         // pinned staging of the header message
    uint8_t *h_small;                       // pinned: [0,16) tag_h  [16,20) status_h  [32,44) nonce_h  [48,64) expected tag_h
    uint8_t *d_hdr;                         // device: the header message, processed in place
    uint8_t *d_small;                       // device: [0,16) AAD_H  [16,32) tag_h  [32,36) status_h  [64,72) DATASUM accumulator
    gcm_ctx *g[2];                          // cached key contexts: 0 Header Key, 1 Data Key
    uint8_t key[2][32];
    int key_bits[2];
};

namespace {

#define CUF(call)                                                                                  \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess) return fail(res, gcm_cuda_fail(e__), cudaGetErrorString(e__));     \
    } while (0)

int fail(FitsOperationResult *res, int code, const char *msg)
{
    if (res) {
        res->error_code = code;
        snprintf(res->error_message, sizeof res->error_message, "%s", msg);
    }
    return code;
}

void wipe_host(void *p, size_t n)
{
    memset(p, 0, n);
    __asm__ __volatile__("" : : "r"(p) : "memory");
}

// the key context of slot `which`, rebuilt only when the key changes (the setup kernel runs once per key)
int ensure_key(gfc_context *c, int which, const uint8_t *key, int key_bits)
{
    if (c->g[which] && c->key_bits[which] == key_bits && memcmp(c->key[which], key, key_bits / 8) == 0) return GCM_OK;
    if (c->g[which]) gcm_destroy(c->g[which]);
    c->g[which] = nullptr;
    int rc = gcm_init_on_device(&c->g[which], key, key_bits, c->device);
    if (rc != GCM_OK) return rc;
    memcpy(c->key[which], key, key_bits / 8);
    c->key_bits[which] = key_bits;
    return GCM_OK;
}

bool draw_nonce(uint8_t out[12])           // the host system's entropy pool
{
    FILE *f = fopen("/dev/urandom", "rb");
    if (!f) return false;
    const bool ok = fread(out, 1, 12, f) == 12;
    fclose(f);
    return ok;
}

struct Orig {                              // ORIG_BITPIX, ORIG_NAXIS, ORIG_NAXISn (L121, footnote 3)
    long long bitpix = 0, naxis = 0, dim[9] = {0};
};

bool read_orig(const Header &h, const char *kb, const char *kn, const char *kd_fmt, Orig *o)
{
    if (!get_int(h, kb, &o->bitpix) || !get_int(h, kn, &o->naxis) || o->naxis < 0 || o->naxis > 9) return false;
    for (int i = 0; i < o->naxis; i++) {
        char k[32];
        snprintf(k, sizeof k, kd_fmt, i + 1);
        if (!get_int(h, k, &o->dim[i]) || o->dim[i] < 0) return false;
    }
    return true;
}

// L151-L155: AAD_Data = NONCE_D || Serialize(ORIG_BITPIX) || Serialize(ORIG_NAXIS) || ..., Serialize = strict
// ASCII decimal, plain concatenation (reading F6)
std::string data_aad(const uint8_t nonce_d[12], const Orig &o)
{
    std::string a((const char *)nonce_d, 12);
    a += std::to_string(o.bitpix);
    a += std::to_string(o.naxis);
    for (int i = 0; i < o.naxis; i++) a += std::to_string(o.dim[i]);
    return a;
}

std::string envelope_header(const uint8_t nonce_h[12], const uint8_t nonce_d[12], const uint8_t tag_h[16],
                            const uint8_t tag_d[16], const Orig &o, const uint8_t *enc_hdr, uint64_t hlen)
{
    std::string h;
    put_logical(h, "SIMPLE", true);
    put_int(h, "BITPIX", 8);
    put_int(h, "NAXIS", 0);
    put_logical(h, "EXTEND", true);
    put_str(h, "LONGSTRN", "OGIP 1.0");
    put_str(h, "NONCE_H", to_hex(nonce_h, 12));
    put_str(h, "NONCE_D", to_hex(nonce_d, 12));
    put_str(h, "AUTHTAGH", to_hex(tag_h, 16));
    put_str(h, "AUTHTAGD", to_hex(tag_d, 16));
    put_int(h, "ORIG_BPX", o.bitpix);
    put_int(h, "ORIG_NAX", o.naxis);
    for (int i = 0; i < o.naxis; i++) {
        char k[32];
        snprintf(k, sizeof k, "ORIG_NA%d", i + 1);
        put_int(h, k, o.dim[i]);
    }
    put_long_str(h, "ENCHDR", to_hex(enc_hdr, hlen));
    return h;
}

std::string bintable_header(uint64_t n)
{
    std::string h;
    put_str(h, "XTENSION", "BINTABLE");
    put_int(h, "BITPIX", 8);
    put_int(h, "NAXIS", 2);
    put_int(h, "NAXIS1", (long long)n);
    put_int(h, "NAXIS2", 1);
    put_int(h, "PCOUNT", 0);
    put_int(h, "GCOUNT", 1);
    put_int(h, "TFIELDS", 1);
    put_str(h, "TTYPE1", "ENCDATA");
    put_str(h, "TFORM1", std::to_string(n) + "B");       // L125: TFORM = '<N>B'
    put_str(h, "EXTNAME", "ENCDATA");
    return h;
}

std::string minimal_header(const Orig &o)                 // L241: header fallback (reading F9)
{
    std::string h;
    put_logical(h, "SIMPLE", true);
    put_int(h, "BITPIX", o.bitpix);
    put_int(h, "NAXIS", o.naxis);
    for (int i = 0; i < o.naxis; i++) {
        char k[32];
        snprintf(k, sizeof k, "NAXIS%d", i + 1);
        put_int(h, k, o.dim[i]);
    }
    put_end_and_pad(h);
    return h;
}

uint64_t header_length_with_checksums(uint64_t card_bytes)     // + DATASUM, CHECKSUM, END, padding
{
    return (card_bytes + 3 * kCard + kBlock - 1) / kBlock * kBlock;
}

void reset_result(FitsOperationResult *res)
{
    memset(res, 0, sizeof *res);
}

}  // namespace

// ---- C ABI ----------------------------------------------------------------------------------------------
extern "C" int gfc_context_create(gfc_context **out, uint64_t max_header_bytes, uint64_t max_data_bytes)
{
    if (!out) return GCM_ERR_ARG;
    *out = nullptr;
    if (max_header_bytes < kBlock) max_header_bytes = kBlock;
    if (max_header_bytes > (1ull << 30) || max_data_bytes > (1ull << 36) - 32) return GCM_ERR_LEN;
    gfc_context *c = new (std::nothrow) gfc_context;
    if (!c) return GCM_ERR_NOMEM;
    memset(c, 0, sizeof *c);
    c->max_header = (max_header_bytes + kBlock - 1) / kBlock * kBlock;
    c->max_data = max_data_bytes;
    // container = envelope header (hex ENCHDR: 160 card bytes per 67 hex characters) + BINTABLE header + payload
    c->out_cap = 5 * c->max_header + c->max_data + 16 * kBlock;
    // the library's one notion of "the device": gcm_set_device's choice, else the caller's current device
    cudaError_t e = cudaSuccess;
    int rc_dev = gcm_default_device(&c->device);
    if (rc_dev != GCM_OK) { delete c; return rc_dev; }
    DeviceGuard guard(c->device);
    e = guard.err;
    do {
        if (e != cudaSuccess) break;
        if ((e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device)) != cudaSuccess) break;
        if ((e = cudaStreamCreateWithFlags(&c->streamH, cudaStreamNonBlocking)) != cudaSuccess) break;
        if ((e = cudaStreamCreateWithFlags(&c->streamD, cudaStreamNonBlocking)) != cudaSuccess) break;
        if ((e = cudaEventCreate(&c->evH0)) != cudaSuccess) break;
        if ((e = cudaEventCreate(&c->evH1)) != cudaSuccess) break;
        if ((e = cudaEventCreate(&c->evD0)) != cudaSuccess) break;
        if ((e = cudaEventCreate(&c->evD1)) != cudaSuccess) break;
        if ((e = cudaHostAlloc((void **)&c->h_out, c->out_cap, cudaHostAllocDefault)) != cudaSuccess) break;
        if ((e = cudaHostAlloc((void **)&c->h_hdr, c->max_header, cudaHostAllocDefault)) != cudaSuccess) break;
        if ((e = cudaHostAlloc((void **)&c->h_small, 128, cudaHostAllocDefault)) != cudaSuccess) break;
        if ((e = cudaMalloc((void **)&c->d_hdr, c->max_header)) != cudaSuccess) break;
        if ((e = cudaMalloc((void **)&c->d_small, 128)) != cudaSuccess) break;
        e = cudaMemset(c->d_small, 0, 128);
    } while (0);
    if (e != cudaSuccess) {
        gfc_context_destroy(c);
        return gcm_cuda_fail(e);
    }
    *out = c;
    return GCM_OK;
}

extern "C" void gfc_context_destroy(gfc_context *c)
{
    if (!c) return;
    DeviceGuard guard(c->device);
    if (c->streamH) cudaStreamSynchronize(c->streamH);
    if (c->streamD) cudaStreamSynchronize(c->streamD);
    for (int i = 0; i < 2; i++) {
        if (c->g[i]) gcm_destroy(c->g[i]);
        wipe_host(c->key[i], sizeof c->key[i]);
    }
    if (c->d_hdr) { cudaMemset(c->d_hdr, 0, c->max_header); cudaFree(c->d_hdr); }
    if (c->d_small) cudaFree(c->d_small);
    if (c->h_hdr) { wipe_host(c->h_hdr, c->max_header); cudaFreeHost(c->h_hdr); }
    if (c->h_small) cudaFreeHost(c->h_small);
    if (c->h_out) cudaFreeHost(c->h_out);
    if (c->evH0) cudaEventDestroy(c->evH0);
    if (c->evH1) cudaEventDestroy(c->evH1);
    if (c->evD0) cudaEventDestroy(c->evD0);
    if (c->evD1) cudaEventDestroy(c->evD1);
    if (c->streamH) cudaStreamDestroy(c->streamH);
    if (c->streamD) cudaStreamDestroy(c->streamD);
    delete c;
}

extern "C" int gfc_encrypt_frame(gfc_context *c, const uint8_t *fits, uint64_t fits_len,
                                 const uint8_t *key_h, const uint8_t *key_d, int key_bits,
                                 const uint8_t *nonce_h_in, const uint8_t *nonce_d_in, FitsOperationResult *res)
{
    if (!res) return GCM_ERR_ARG;
    reset_result(res);
    if (!c || !fits || !key_h || !key_d || (key_bits != 128 && key_bits != 256)) return fail(res, GCM_ERR_ARG, "bad argument");
    Header hd;
    Orig o;
    if (!parse_header(fits, fits_len, 0, &hd) || !read_orig(hd, "BITPIX", "NAXIS", "NAXIS%d", &o))
        return fail(res, GFC_ERR_FORMAT, "not a FITS file: primary header without END / BITPIX / NAXIS");
    const uint64_t hlen = hd.length, n = fits_len - hlen;
    if (hlen > c->max_header || n > c->max_data) return fail(res, GFC_ERR_CAPACITY, "file larger than the context was created for");
    DeviceGuard guard(c->device);
    CUF(guard.err);
    int rc = ensure_key(c, 0, key_h, key_bits);
    if (rc == GCM_OK) rc = ensure_key(c, 1, key_d, key_bits);
    if (rc != GCM_OK) return fail(res, rc, "key setup failed");
    uint8_t nonce_h[12], nonce_d[12];
    if (nonce_h_in) memcpy(nonce_h, nonce_h_in, 12);
    else if (!draw_nonce(nonce_h)) return fail(res, GCM_ERR_ARG, "no entropy source for NONCE_H");
    if (nonce_d_in) memcpy(nonce_d, nonce_d_in, 12);
    else if (!draw_nonce(nonce_d)) return fail(res, GCM_ERR_ARG, "no entropy source for NONCE_D");

    // ---- streamH: the header message (L214), asynchronous
    memcpy(c->h_hdr, fits, hlen);
    memcpy(c->h_small + 32, nonce_h, 12);
    CUF(cudaEventRecord(c->evH0, c->streamH));
    CUF(cudaMemcpyAsync(c->d_hdr, c->h_hdr, hlen, cudaMemcpyHostToDevice, c->streamH));
    CUF(cudaMemcpyAsync(c->d_small, c->h_small + 32, 12, cudaMemcpyHostToDevice, c->streamH));   // AAD_H = NONCE_H (F7)
    rc = gcm_encrypt_async(c->g[0], nonce_h, c->d_small, 12, c->d_hdr, hlen, c->d_hdr, c->d_small + 16, c->streamH);
    if (rc != GCM_OK) return fail(res, rc, "header message launch failed");
    CUF(cudaMemcpyAsync(c->h_hdr, c->d_hdr, hlen, cudaMemcpyDeviceToHost, c->streamH));
    CUF(cudaMemcpyAsync(c->h_small, c->d_small + 16, 16, cudaMemcpyDeviceToHost, c->streamH));
    CUF(cudaEventRecord(c->evH1, c->streamH));

    // ---- layout: both header lengths are known before any ciphertext exists
    uint8_t zero16[16] = {0};
    const uint64_t L0 = header_length_with_checksums(envelope_header(nonce_h, nonce_d, zero16, zero16, o, c->h_hdr, 0).size() +
                                                     ((2 * hlen + 66) / 67 - 1) * kCard);
    const uint64_t L1 = header_length_with_checksums(bintable_header(n).size());
    const uint64_t n_pad = (n + kBlock - 1) / kBlock * kBlock;
    const uint64_t total = L0 + L1 + n_pad;
    if (total > c->out_cap) return fail(res, GFC_ERR_CAPACITY, "container larger than the result buffer");

    // ---- streamD: the data message (L215-L217), chunked H2D -> fused AES-GCM kernel -> DATASUM kernel -> D2H
    unsigned long long *d_sum = (unsigned long long *)(c->d_small + 64);
    uint8_t tag_d[16];
    const std::string aad = data_aad(nonce_d, o);
    CUF(cudaMemsetAsync(d_sum, 0, 8, c->streamD));
    CUF(cudaEventRecord(c->evD0, c->streamD));
    {
        CtxLock lock(c->g[1]);                  // gcm_host_run wants the key context's lock held (one call at a time)
        if (!lock.ok) return fail(res, GCM_ERR_BUSY, "data key context is in use");
        rc = gcm_host_run(c->g[1], MODE_ENCRYPT, nonce_d, aad.data(), aad.size(), fits + hlen, n, c->h_out + L0 + L1, tag_d,
                          c->streamD, d_sum);
    }
    if (rc != GCM_OK) return fail(res, rc, "data message failed");
    CUF(cudaMemcpyAsync(c->h_small + 64, d_sum, 8, cudaMemcpyDeviceToHost, c->streamD));
    CUF(cudaEventRecord(c->evD1, c->streamD));
    CUF(cudaStreamSynchronize(c->streamD));
    CUF(cudaStreamSynchronize(c->streamH));
    unsigned long long acc;
    memcpy(&acc, c->h_small + 64, 8);
    memset(c->h_out + L0 + L1 + n, 0, n_pad - n);

    // ---- the two headers
    std::string h0 = envelope_header(nonce_h, nonce_d, c->h_small, tag_d, o, c->h_hdr, hlen);
    finish_header(h0, 0);
    std::string h1 = bintable_header(n);
    finish_header(h1, fits_sum_fold(acc));
    if (h0.size() != L0 || h1.size() != L1) return fail(res, GCM_ERR_ARG, "internal: header length mismatch");
    memcpy(c->h_out, h0.data(), L0);
    memcpy(c->h_out + L0, h1.data(), L1);
    cudaEventElapsedTime(&res->header_ms, c->evH0, c->evH1);
    cudaEventElapsedTime(&res->data_ms, c->evD0, c->evD1);
    res->data_buffer = c->h_out;
    res->buffer_size = total;
    return GCM_OK;
}

extern "C" int gfc_decrypt_frame(gfc_context *c, const uint8_t *ctr, uint64_t len,
                                 const uint8_t *key_h, const uint8_t *key_d, int key_bits, FitsOperationResult *res)
{
    if (!res) return GCM_ERR_ARG;
    reset_result(res);
    if (!c || !ctr || ((key_h || key_d) && key_bits != 128 && key_bits != 256)) return fail(res, GCM_ERR_ARG, "bad argument");
    // ---- HDU 0: the envelope
    Header h0, h1;
    Orig o;
    long long naxis0 = -1, n_ll = -1;
    std::string s_nh, s_nd, s_th, s_td, s_enc, s_xt;
    uint8_t nonce_h[12], nonce_d[12], tag_h[16], tag_d[16];
    if (!parse_header(ctr, len, 0, &h0) || !get_int(h0, "NAXIS", &naxis0) || naxis0 != 0)
        return fail(res, GFC_ERR_FORMAT, "HDU 0 is not a metadata-only primary HDU");
    if (!get_str(h0, "NONCE_H", &s_nh) || !from_hex(s_nh, nonce_h, 12) || !get_str(h0, "NONCE_D", &s_nd) ||
        !from_hex(s_nd, nonce_d, 12) || !get_str(h0, "AUTHTAGH", &s_th) || !from_hex(s_th, tag_h, 16) ||
        !get_str(h0, "AUTHTAGD", &s_td) || !from_hex(s_td, tag_d, 16) || !get_str(h0, "ENCHDR", &s_enc) ||
        s_enc.empty() || (s_enc.size() & 1))
        return fail(res, GFC_ERR_FORMAT, "envelope keyword missing or malformed");
    if (!read_orig(h0, "ORIG_BPX", "ORIG_NAX", "ORIG_NA%d", &o)) return fail(res, GFC_ERR_FORMAT, "ORIG_* keywords missing");
    const uint64_t hlen = s_enc.size() / 2;
    if (hlen > c->max_header) return fail(res, GFC_ERR_CAPACITY, "header larger than the context was created for");
    if (!from_hex(s_enc, c->h_hdr, hlen)) return fail(res, GFC_ERR_FORMAT, "ENCHDR is not hex text");
    // ---- HDU 1: the data container
    if (!parse_header(ctr, len, h0.length, &h1) || !get_str(h1, "XTENSION", &s_xt) || s_xt != "BINTABLE" ||
        !get_int(h1, "NAXIS1", &n_ll) || n_ll < 0)
        return fail(res, GFC_ERR_FORMAT, "HDU 1 is not the BINTABLE data container");
    const uint64_t n = (uint64_t)n_ll, d_off = h0.length + h1.length;
    if (d_off + n > len) return fail(res, GFC_ERR_FORMAT, "truncated payload");
    if (n > c->max_data) return fail(res, GFC_ERR_CAPACITY, "payload larger than the context was created for");
    const std::string fb = minimal_header(o);
    const uint64_t room = hlen > fb.size() ? hlen : fb.size();     // the payload lands behind the larger header
    if (room + n > c->out_cap) return fail(res, GFC_ERR_CAPACITY, "result larger than the result buffer");
    DeviceGuard guard(c->device);
    CUF(guard.err);

    // ---- streamH: ENCHDR (L214); no Header Key -> nothing to do, the fallback header is used (L241)
    bool header_sent = false;
    if (key_h) {
        int rc = ensure_key(c, 0, key_h, key_bits);
        if (rc != GCM_OK) return fail(res, rc, "header key setup failed");
        memcpy(c->h_small + 32, nonce_h, 12);
        memcpy(c->h_small + 48, tag_h, 16);
        CUF(cudaEventRecord(c->evH0, c->streamH));
        CUF(cudaMemcpyAsync(c->d_hdr, c->h_hdr, hlen, cudaMemcpyHostToDevice, c->streamH));
        CUF(cudaMemcpyAsync(c->d_small, c->h_small + 32, 12, cudaMemcpyHostToDevice, c->streamH));
        CUF(cudaMemcpyAsync(c->d_small + 16, c->h_small + 48, 16, cudaMemcpyHostToDevice, c->streamH));
        rc = gcm_decrypt_verify_async(c->g[0], nonce_h, c->d_small, 12, c->d_hdr, hlen, c->d_hdr, c->d_small + 16,
                                      c->d_small + 32, c->streamH);
        if (rc != GCM_OK) return fail(res, rc, "header message launch failed");
        CUF(cudaMemcpyAsync(c->h_hdr, c->d_hdr, hlen, cudaMemcpyDeviceToHost, c->streamH));
        CUF(cudaMemcpyAsync(c->h_small + 16, c->d_small + 32, 4, cudaMemcpyDeviceToHost, c->streamH));
        CUF(cudaEventRecord(c->evH1, c->streamH));
        header_sent = true;
    }
    // ---- streamD: the payload (L215-L219); no Data Key -> suppressed (L243)
    bool payload_ok = false;
    uint8_t *pay = c->h_out + room;
    if (key_d) {
        int rc = ensure_key(c, 1, key_d, key_bits);
        if (rc != GCM_OK) return fail(res, rc, "data key setup failed");
        const std::string aad = data_aad(nonce_d, o);
        CUF(cudaEventRecord(c->evD0, c->streamD));
        {
            CtxLock lock(c->g[1]);
            if (!lock.ok) return fail(res, GCM_ERR_BUSY, "data key context is in use");
            rc = gcm_host_run(c->g[1], MODE_DECRYPT, nonce_d, aad.data(), aad.size(), ctr + d_off, n, pay, tag_d, c->streamD, nullptr);
        }
        if (rc < 0) return fail(res, rc, "data message failed");
        CUF(cudaEventRecord(c->evD1, c->streamD));
        CUF(cudaStreamSynchronize(c->streamD));
        cudaEventElapsedTime(&res->data_ms, c->evD0, c->evD1);
        payload_ok = rc == GCM_OK;             // GCM_ERR_AUTH: gcm_host_run has zero-filled the output
    } else {
        memset(pay, 0, n);
    }
    bool header_ok = false;
    if (header_sent) {
        CUF(cudaStreamSynchronize(c->streamH));
        cudaEventElapsedTime(&res->header_ms, c->evH0, c->evH1);
        int status;
        memcpy(&status, c->h_small + 16, 4);
        header_ok = status == 0;
    }
    uint8_t *start;
    if (header_ok) {
        start = pay - hlen;
        memcpy(start, c->h_hdr, hlen);
    } else {
        start = pay - fb.size();
        memcpy(start, fb.data(), fb.size());
    }
    res->data_buffer = start;
    res->buffer_size = (uint64_t)(pay - start) + n;
    res->warning_code = (header_ok ? 0 : GFC_HEADER_FALLBACK) | (payload_ok ? 0 : GFC_PAYLOAD_SUPPRESSED);
    return GCM_OK;
}
