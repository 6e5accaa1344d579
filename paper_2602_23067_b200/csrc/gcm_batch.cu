// gcm_batch.cu -- batched many-message entry points (include/gcm.h).
//
// Large messages (FITS-sized HDUs, config C3) go through the fused single-message kernel with a
// per-key context that is cached across calls, one launch per message on the caller's stream.
#include <cuda_runtime.h>
#include <string.h>
#include <map>
#include <string>
#include <vector>
#include <mutex>

#include "../../include/gcm.h"
#include "gcm_common.cuh"
#include "gcm_api_internal.h"

namespace {
struct KeyCache {
    std::mutex mu;
    std::map<std::string, gcm_ctx *> by_key;   // key bytes (+ device) -> context
    std::vector<std::string> order;            // insertion order, for eviction
    static constexpr size_t kMax = 64;
};
KeyCache g_cache;

void evict_all_locked()
{
    for (auto &kv : g_cache.by_key) gcm_destroy(kv.second);
    g_cache.by_key.clear();
    for (auto &s : g_cache.order) { volatile char *v = &s[0]; for (size_t i = 0; i < s.size(); i++) v[i] = 0; }
    g_cache.order.clear();
}

int ctx_for_key(const uint8_t *key, int key_bits, gcm_ctx **out)
{
    if (!key || (key_bits != 128 && key_bits != 256)) return GCM_ERR_ARG;
    int dev = 0;
    cudaGetDevice(&dev);
    std::string id((const char *)key, key_bits / 8);
    id.push_back((char)dev);
    auto it = g_cache.by_key.find(id);
    if (it != g_cache.by_key.end()) { *out = it->second; return GCM_OK; }
    if (g_cache.by_key.size() >= KeyCache::kMax) evict_all_locked();
    gcm_ctx *c = nullptr;
    int rc = gcm_init(&c, key, key_bits);
    if (rc != GCM_OK) return rc;
    g_cache.by_key[id] = c;
    g_cache.order.push_back(id);
    *out = c;
    return GCM_OK;
}
}  // namespace

extern "C" void gcm_batch_release(void)
{
    std::lock_guard<std::mutex> lock(g_cache.mu);
    evict_all_locked();
}

static int run_batch(gcm_msg *msgs, uint32_t n, void *stream, bool decrypt)
{
    if (n && !msgs) return GCM_ERR_ARG;
    std::lock_guard<std::mutex> lock(g_cache.mu);
    int first_err = GCM_OK, failures = 0;
    for (uint32_t i = 0; i < n; i++) {
        gcm_msg &m = msgs[i];
        gcm_ctx *c = nullptr;
        int rc = ctx_for_key(m.key, m.key_bits, &c);
        if (rc == GCM_OK) {
            rc = decrypt ? gcm_decrypt_verify(c, m.iv, m.d_aad, m.aad_len, m.d_in, m.len, m.d_out, m.tag, stream)
                         : gcm_encrypt(c, m.iv, m.d_aad, m.aad_len, m.d_in, m.len, m.d_out, m.tag, stream);
        }
        m.status = rc;
        if (rc < 0 && first_err == GCM_OK) first_err = rc;
        if (rc == GCM_ERR_AUTH) failures++;
    }
    if (first_err != GCM_OK) return first_err;
    return decrypt ? failures : GCM_OK;
}

extern "C" int gcm_encrypt_batch(gcm_msg *msgs, uint32_t n, void *stream) { return run_batch(msgs, n, stream, false); }
extern "C" int gcm_decrypt_verify_batch(gcm_msg *msgs, uint32_t n, void *stream) { return run_batch(msgs, n, stream, true); }
