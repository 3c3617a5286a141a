// Time-frame streaming: a time frame is cut into GROUPS OF SECTORS -- sectors
// are independent units from S1 to S7, so a group needs no halo and no exchange -- and every group runs on its own
// context / stream / host thread: load (H2D), tpcca_run, delivery (D2H).  The copies of one group overlap the
// kernels of the others on the copy engines, the first tracks leave the GPU after 1/G of the input has arrived, and
// one workspace holds 1/G of the time frame.  Included at the end of tpcca_api.cu (same translation unit).
#pragma once
#include <condition_variable>
#include <mutex>
#include <thread>

struct tpcca_pipeline {
  int ns = 0, ng = 0, device = 0;
  std::vector<tpcca_ctx*> ctx;          // one context per group
  std::vector<int> first;               // group g owns sectors [first[g], first[g + 1])
  std::vector<float> ms;                // per group: host wall time of its last run [ms]
  std::string err;
};

namespace {
thread_local std::string g_pipe_error;
int pipe_err(tpcca_pipeline* p, int code, const std::string& m) {
  if (p) p->err = m; else g_pipe_error = m;
  return code;
}
}  // namespace

extern "C" {

const char* tpcca_pipeline_last_error(const tpcca_pipeline* p) { return p ? p->err.c_str() : g_pipe_error.c_str(); }

int tpcca_pipeline_workspace_bytes(const tpcca_params* params, int n_groups, int64_t max_clusters_group,
                                   int64_t max_start_hits_group, size_t* out_bytes) {
  if (!params || !out_bytes || n_groups < 1 || n_groups > params->n_sectors)
    return pipe_err(nullptr, TPCCA_E_ARG, "n_groups must be in 1..n_sectors");
  tpcca_params q = *params;
  q.n_sectors = (params->n_sectors + n_groups - 1) / n_groups;      // the largest group
  const int rc = tpcca_workspace_bytes(&q, max_clusters_group, max_start_hits_group, out_bytes);
  if (rc) return pipe_err(nullptr, rc, tpcca_last_error(nullptr));
  return TPCCA_OK;
}

int tpcca_pipeline_create(const tpcca_params* params, int cuda_device, int n_groups, void* const* cuda_streams,
                          void* const* workspaces, size_t workspace_bytes_each, int64_t max_clusters_group,
                          int64_t max_start_hits_group, tpcca_pipeline** out) {
  if (!out) return pipe_err(nullptr, TPCCA_E_ARG, "out is NULL");
  *out = nullptr;
  if (!params || !cuda_streams || !workspaces || n_groups < 1 || n_groups > params->n_sectors)
    return pipe_err(nullptr, TPCCA_E_ARG, "bad arguments (n_groups must be in 1..n_sectors)");
  tpcca_pipeline* p = new tpcca_pipeline;
  p->ns = params->n_sectors; p->ng = n_groups; p->device = cuda_device;
  p->first.resize(n_groups + 1);
  for (int g = 0; g <= n_groups; ++g) p->first[g] = (int)((int64_t)g * p->ns / n_groups);
  p->ms.assign(n_groups, 0.f);
  for (int g = 1; g < n_groups; ++g)
    for (int h = 0; h < g; ++h)
      if (cuda_streams[g] == cuda_streams[h]) {      // any two groups on one stream would run one after the other
        tpcca_pipeline_destroy(p);
        return pipe_err(nullptr, TPCCA_E_ARG, "every group needs its own stream (groups " + std::to_string(h) + " and " +
                                              std::to_string(g) + " share one)");
      }
  for (int g = 0; g < n_groups; ++g) {
    tpcca_params q = *params;
    q.n_sectors = p->first[g + 1] - p->first[g];
    tpcca_ctx* c = nullptr;
    const int rc = tpcca_create(&q, cuda_device, cuda_streams[g], workspaces[g], workspace_bytes_each, max_clusters_group,
                                max_start_hits_group, &c);
    if (rc) {
      const std::string m = std::string("group ") + std::to_string(g) + ": " + tpcca_last_error(nullptr);
      tpcca_pipeline_destroy(p);
      return pipe_err(nullptr, rc, m);
    }
    p->ctx.push_back(c);
  }
  *out = p;
  return TPCCA_OK;
}

int tpcca_pipeline_run(tpcca_pipeline* p, const int64_t* n, const float* const* y, const float* const* z,
                       const uint16_t* const* row, int mem_space, uint32_t stage_mask, uint32_t what,
                       tpcca_tracks_view* views) {
  if (!p || !n || !y || !z || !row || !views) return pipe_err(p, TPCCA_E_ARG, "NULL argument");
  // S8 links tracks ACROSS sectors; a group is a context of its own with group-local sector numbers, so it would
  // miss every link over a group boundary and number the others wrongly.  Refused instead of delivered wrong.
  if ((stage_mask & TPCCA_STAGE_MERGE) || (what & TPCCA_OUT_MERGE))
    return pipe_err(p, TPCCA_E_ARG, "the pipeline runs sector groups independently: TPCCA_STAGE_MERGE / TPCCA_OUT_MERGE "
                                    "(cross-sector merging) need one context over all sectors (tpcca_run)");
  std::vector<int> rc(p->ng, TPCCA_OK);
  std::vector<std::string> msg(p->ng);
  // the groups issue their loads in group order (group g + 1 queues its H2D copies after group g), so the copy
  // engine serves them one after the other and group 0 starts computing after 1 / G of the input
  std::mutex mu;
  std::condition_variable cv;
  int loaded = 0;
  auto work = [&](int g) {
    const auto t0 = std::chrono::steady_clock::now();
    tpcca_ctx* c = p->ctx[g];
    const int s0 = p->first[g], s1 = p->first[g + 1];
    {
      std::unique_lock<std::mutex> lk(mu);
      cv.wait(lk, [&] { return loaded == g; });
    }
    int r = tpcca_reset(c);
    for (int s = s0; s < s1 && !r; ++s) r = tpcca_load_clusters(c, s - s0, n[s], nullptr, y[s], z[s], nullptr, row[s], mem_space);
    {
      std::lock_guard<std::mutex> lk(mu);
      loaded = g + 1;
    }
    cv.notify_all();
    if (!r) r = tpcca_run(c, stage_mask);
    if (!r) r = tpcca_get_tracks_all(c, TPCCA_MEM_HOST, what, views + s0);
    if (r) { rc[g] = r; msg[g] = tpcca_last_error(c); }
    p->ms[g] = std::chrono::duration<float, std::milli>(std::chrono::steady_clock::now() - t0).count();
  };
  std::vector<std::thread> th;
  for (int g = 1; g < p->ng; ++g) th.emplace_back(work, g);
  work(0);
  for (auto& t : th) t.join();
  for (int g = 0; g < p->ng; ++g)
    if (rc[g]) return pipe_err(p, rc[g], std::string("group ") + std::to_string(g) + ": " + msg[g]);
  return TPCCA_OK;
}

int tpcca_pipeline_get_groups(const tpcca_pipeline* p, int32_t* first_sector /*[n_groups + 1]*/, float* ms /*[n_groups]*/) {
  if (!p) return TPCCA_E_ARG;
  for (int g = 0; g <= p->ng && first_sector; ++g) first_sector[g] = p->first[g];
  for (int g = 0; g < p->ng && ms; ++g) ms[g] = p->ms[g];
  return p->ng;
}

void tpcca_pipeline_destroy(tpcca_pipeline* p) {
  if (!p) return;
  for (tpcca_ctx* c : p->ctx) tpcca_destroy(c);
  delete p;
}

}  // extern "C"
