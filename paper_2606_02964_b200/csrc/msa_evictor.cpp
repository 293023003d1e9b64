// Computational-aware block evictor (include/msa_evictor.h): Algorithm 1 of the paper with two ordered
// sets keyed by the time-independent part of the log weight of each branch of Eq. (9).  Host only.
#include "../../include/msa_evictor.h"

#include <algorithm>
#include <cmath>
#include <limits>
#include <new>
#include <set>
#include <unordered_map>
#include <utility>

#include "../../include/msa.h"

namespace {

struct Entry {
    double key1, key2;     // last/alpha + ln dT ;  (last + tau0)/beta + ln dT
};

using Key = std::pair<double, int64_t>;   // (key, block id): ties broken by id, deterministically

}  // namespace

struct msa_evictor_s {
    msa_evictor_config cfg{};
    double ln_lambda = 0.0;
    std::set<Key> bt1, bt2;
    std::unordered_map<int64_t, Entry> blocks;

    double log_w1(const Entry &e, double t) const { return e.key1 - t / cfg.alpha; }
    double log_w2(const Entry &e, double t) const { return ln_lambda + e.key2 - t / cfg.beta; }
    void erase(int64_t id, const Entry &e)
    {
        bt1.erase(Key(e.key1, id));
        bt2.erase(Key(e.key2, id));
        blocks.erase(id);
    }
};

extern "C" {

int msa_evictor_create(const msa_evictor_config *cfg, msa_evictor *out)
{
    if (!cfg || !out) return MSA_ERR_INVALID_ARG;
    if (!(cfg->alpha > 0.0) || !(cfg->beta > 0.0) || !(cfg->tau0 >= 0.0) || !(cfg->lambda > 0.0)) return MSA_ERR_INVALID_ARG;
    if (!std::isfinite(cfg->k5) || !std::isfinite(cfg->c0) || cfg->k5 < 0.0) return MSA_ERR_INVALID_ARG;
    msa_evictor_s *ev = new (std::nothrow) msa_evictor_s();
    if (!ev) return MSA_ERR_INVALID_ARG;
    ev->cfg = *cfg;
    ev->ln_lambda = std::log(cfg->lambda);
    *out = ev;
    return MSA_OK;
}

void msa_evictor_destroy(msa_evictor ev) { delete ev; }

int msa_evictor_add(msa_evictor ev, int64_t block_id, int64_t position, double last_access)
{
    if (!ev || position < 0 || !std::isfinite(last_access)) return MSA_ERR_INVALID_ARG;
    const double dT = 2.0 * ev->cfg.k5 * static_cast<double>(position) + ev->cfg.c0;
    if (!(dT > 0.0)) return MSA_ERR_INVALID_ARG;
    if (ev->blocks.count(block_id)) return MSA_ERR_OVERLAP;
    const double ln_dT = std::log(dT);
    Entry e;
    e.key1 = last_access / ev->cfg.alpha + ln_dT;
    e.key2 = (last_access + ev->cfg.tau0) / ev->cfg.beta + ln_dT;
    ev->blocks.emplace(block_id, e);
    ev->bt1.insert(Key(e.key1, block_id));
    ev->bt2.insert(Key(e.key2, block_id));
    return MSA_OK;
}

int msa_evictor_remove(msa_evictor ev, int64_t block_id)
{
    if (!ev) return MSA_ERR_INVALID_ARG;
    auto it = ev->blocks.find(block_id);
    if (it == ev->blocks.end()) return MSA_ERR_OUT_OF_RANGE;
    const Entry e = it->second;
    ev->erase(block_id, e);
    return MSA_OK;
}

int msa_evictor_evict(msa_evictor ev, double t_now, int64_t *block_id)
{
    if (!ev || !block_id) return MSA_ERR_INVALID_ARG;
    if (ev->blocks.empty()) return MSA_ERR_OUT_OF_RANGE;
    const Key b1 = *ev->bt1.begin(), b2 = *ev->bt2.begin();
    const double w1 = b1.first - t_now / ev->cfg.alpha;
    const double w2 = ev->ln_lambda + b2.first - t_now / ev->cfg.beta;
    const int64_t victim = (w1 <= w2) ? b1.second : b2.second;       // Algorithm 1 line 8 (in the log domain)
    const Entry e = ev->blocks[victim];
    ev->erase(victim, e);
    *block_id = victim;
    return MSA_OK;
}

int msa_evictor_evict_linear(msa_evictor ev, double t_now, int64_t *block_id)
{
    if (!ev || !block_id) return MSA_ERR_INVALID_ARG;
    if (ev->blocks.empty()) return MSA_ERR_OUT_OF_RANGE;
    // the same argmin, found the O(n) way: first the smallest w1, then the smallest lambda*w2 (ties by id)
    double best1 = std::numeric_limits<double>::infinity(), best2 = best1;
    int64_t id1 = 0, id2 = 0;
    for (const auto &kv : ev->blocks) {
        const double a = ev->log_w1(kv.second, t_now), b = ev->log_w2(kv.second, t_now);
        if (a < best1 || (a == best1 && kv.first < id1)) { best1 = a; id1 = kv.first; }
        if (b < best2 || (b == best2 && kv.first < id2)) { best2 = b; id2 = kv.first; }
    }
    const int64_t victim = (best1 <= best2) ? id1 : id2;
    const Entry e = ev->blocks[victim];
    ev->erase(victim, e);
    *block_id = victim;
    return MSA_OK;
}

int msa_evictor_set_lambda(msa_evictor ev, double lambda)
{
    if (!ev || !(lambda > 0.0)) return MSA_ERR_INVALID_ARG;
    ev->cfg.lambda = lambda;
    ev->ln_lambda = std::log(lambda);
    return MSA_OK;
}

int64_t msa_evictor_size(msa_evictor ev) { return ev ? static_cast<int64_t>(ev->blocks.size()) : 0; }

double msa_evictor_weight(msa_evictor ev, int64_t block_id, double t_now)
{
    if (!ev) return std::numeric_limits<double>::quiet_NaN();
    auto it = ev->blocks.find(block_id);
    if (it == ev->blocks.end()) return std::numeric_limits<double>::quiet_NaN();
    return std::exp(std::min(ev->log_w1(it->second, t_now), ev->log_w2(it->second, t_now)));
}

}  // extern "C"
