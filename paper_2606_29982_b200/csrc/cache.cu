// cache.cu — LFU expert cache of the offloading system (Fig. 8; SURVEY.md §8(f)
// NEXT-1): host-side state shared by the layers attached to it.  The paper names the policy
// only; the rules are readings R30-R34 of DESIGN.md §3 (restated at the declaration in
// include/caee.h).  The device side of a miss (the H2D copy into the slot chosen here, overlapped
// with the hits' compute) is forward_impl's offload path in caee_api.cu.
#include <new>

#include "caee_internal.cuh"

namespace {
std::string g_cache_err;
}

extern "C" {

caee_status caee_cache_create(int32_t n_slots, caee_cache** out) {
  if (!out) return CAEE_EINVAL;
  *out = nullptr;
  if (n_slots <= 0 || n_slots > (1 << 20)) return CAEE_EINVAL;
  caee_cache* k = new (std::nothrow) caee_cache();
  if (!k) return CAEE_ENOMEM;
  k->n_slots = n_slots;
  cudaGetDevice(&k->device);
  k->slot_ptr.assign(n_slots, nullptr);
  k->slot_layer.assign(n_slots, -1);
  k->slot_expert.assign(n_slots, -1);
  *out = k;
  return CAEE_OK;
}

void caee_cache_destroy(caee_cache* k) {
  if (!k) return;
  for (caee_ctx* c : k->layers)
    if (c) { c->cache = nullptr; c->cache_layer = -1; c->have_weights = false; }
  int dev = 0;
  cudaGetDevice(&dev);
  cudaSetDevice(k->device);
  cudaDeviceSynchronize();
  for (uint8_t* p : k->slot_ptr)
    if (p) cudaFree(p);
  cudaSetDevice(dev);
  delete k;
}

caee_status caee_cache_attach(caee_cache* k, caee_ctx* c, int32_t layer_id) {
  if (!c) return CAEE_EINVAL;
  if (!k) return caee_fail(c, CAEE_EINVAL, "cache is NULL");
  if (layer_id < 0 || layer_id >= 4096) return caee_fail(c, CAEE_EINVAL, "layer_id must be in 0..4095");
  if (c->cache) return caee_fail(c, CAEE_ESTATE, "the context is already attached to a cache");
  if (c->kernel != CAEE_KERNEL_UMMA) return caee_fail(c, CAEE_EUNSUPPORTED, "the expert cache needs the UMMA expert kernels (packed images)");
  if (c->device != k->device) return caee_fail(c, CAEE_EINVAL, "cache and context are on different devices");
  if ((size_t)layer_id < k->layers.size() && k->layers[layer_id]) return caee_fail(c, CAEE_ESTATE, "layer %d is already attached", layer_id);
  if (k->layers.size() <= (size_t)layer_id) {
    k->layers.resize(layer_id + 1, nullptr);
    k->freq.resize(layer_id + 1);
    k->slot_of.resize(layer_id + 1);
  }
  k->layers[layer_id] = c;
  k->freq[layer_id].assign(c->d.E, 0);
  k->slot_of[layer_id].assign(c->d.E, -1);
  c->cache = k;
  c->cache_layer = layer_id;
  c->have_weights = false;                       // images move to pinned host memory: set the weights (again)
  c->resident_h.assign(c->d.E, 0);               // R34: the cache starts empty
  return CAEE_OK;
}

caee_status caee_cache_read_stats(const caee_cache* k, caee_cache_stats* out) {
  if (!k || !out) return CAEE_EINVAL;
  *out = k->st;
  return CAEE_OK;
}

caee_status caee_cache_snapshot(const caee_cache* k, int32_t* layer, int32_t* expert, int64_t* freq) {
  if (!k || !layer || !expert || !freq) return CAEE_EINVAL;
  for (int s = 0; s < k->n_slots; ++s) {
    layer[s] = k->slot_layer[s];
    expert[s] = k->slot_expert[s];
    freq[s] = k->slot_layer[s] >= 0 ? k->freq[k->slot_layer[s]][k->slot_expert[s]] : 0;
  }
  return CAEE_OK;
}

}  // extern "C"

// caee_set_weights of an attached layer: the slots exist from the first layer on and every layer
// must have the same packed expert size.
caee_status caee_cache_prepare_layer(caee_ctx* c, size_t slot_bytes) {
  caee_cache* k = c->cache;
  if (k->slot_bytes == 0) {
    k->slot_bytes = slot_bytes;
    for (int s = 0; s < k->n_slots; ++s) CAEE_CUDA(c, cudaMalloc((void**)&k->slot_ptr[s], slot_bytes));
  } else if (k->slot_bytes != slot_bytes) {
    return caee_fail(c, CAEE_ESHAPE, "packed expert size %zu differs from the cache's slot size %zu", slot_bytes, k->slot_bytes);
  }
  // (re)setting the weights of a layer drops its keys from the cache
  const int l = c->cache_layer;
  for (int s = 0; s < k->n_slots; ++s)
    if (k->slot_layer[s] == l) { k->slot_layer[s] = -1; k->slot_expert[s] = -1; }
  k->slot_of[l].assign(c->d.E, -1);
  c->resident_h.assign(c->d.E, 0);
  return CAEE_OK;
}

void caee_cache_detach(caee_ctx* c) {
  caee_cache* k = c->cache;
  if (!k) return;
  const int l = c->cache_layer;
  for (int s = 0; s < k->n_slots; ++s)
    if (k->slot_layer[s] == l) { k->slot_layer[s] = -1; k->slot_expert[s] = -1; }
  k->layers[l] = nullptr;
  c->cache = nullptr;
  c->cache_layer = -1;
}

// One step of layer c (R32).  executed: the routed experts of the step's run list, ascending and
// unique.  Counts them, then gives every miss a slot (lowest free slot, else the least frequently
// used key not executed by this step, ties to the smaller (layer, expert)); miss_slots receives
// the slot pointer of each miss in order.  Host state of the evicted keys' layers is updated here;
// their device tables are refreshed at the start of their next step.
caee_status caee_cache_step(caee_ctx* c, const int32_t* executed, int n_executed, std::vector<uint8_t*>* miss_slots) {
  caee_cache* k = c->cache;
  const int l = c->cache_layer;
  std::vector<int64_t>& f = k->freq[l];
  std::vector<int32_t>& so = k->slot_of[l];
  std::vector<uint8_t> in_use(c->d.E, 0);
  for (int i = 0; i < n_executed; ++i) in_use[executed[i]] = 1;
  miss_slots->clear();
  // a step that does not fit fails before anything changes: every miss needs a slot that is free
  // or holds a key this step does not execute
  int n_miss = 0, n_avail = 0;
  for (int i = 0; i < n_executed; ++i) n_miss += so[executed[i]] < 0;
  for (int s = 0; s < k->n_slots; ++s) n_avail += !(k->slot_layer[s] == l && in_use[k->slot_expert[s]]);
  if (n_miss > n_avail)
    return caee_fail(c, CAEE_ESTATE, "the step executes %d experts of layer %d: they do not fit the cache's %d slots", n_executed, l, k->n_slots);
  for (int i = 0; i < n_executed; ++i) ++f[executed[i]];
  for (int i = 0; i < n_executed; ++i) {
    const int e = executed[i];
    if (so[e] >= 0) { ++k->st.hits; continue; }
    ++k->st.misses;
    k->st.h2d_bytes += (int64_t)k->slot_bytes;
    int slot = -1;
    for (int s = 0; s < k->n_slots && slot < 0; ++s)
      if (k->slot_layer[s] < 0) slot = s;
    if (slot < 0) {
      int64_t bf = 0;
      for (int s = 0; s < k->n_slots; ++s) {
        const int sl = k->slot_layer[s], se = k->slot_expert[s];
        if (sl == l && in_use[se]) continue;
        const int64_t sf = k->freq[sl][se];
        const bool better = slot < 0 || sf < bf ||
                            (sf == bf && (sl < k->slot_layer[slot] || (sl == k->slot_layer[slot] && se < k->slot_expert[slot])));
        if (better) { slot = s; bf = sf; }
      }
      if (slot < 0) return caee_fail(c, CAEE_ESTATE, "the step executes %d experts of layer %d: they do not fit the cache's %d slots", n_executed, l, k->n_slots);
      const int vl = k->slot_layer[slot], ve = k->slot_expert[slot];
      k->slot_of[vl][ve] = -1;
      caee_ctx* vc = k->layers[vl];
      if (vc) { vc->resident_h[ve] = 0; if ((size_t)ve < vc->dptr_h.size()) vc->dptr_h[ve] = nullptr; }
      ++k->st.evictions;
    }
    k->slot_layer[slot] = l;
    k->slot_expert[slot] = e;
    so[e] = slot;
    c->resident_h[e] = 1;
    c->dptr_h[e] = k->slot_ptr[slot];
    miss_slots->push_back(k->slot_ptr[slot]);
  }
  return CAEE_OK;
}
