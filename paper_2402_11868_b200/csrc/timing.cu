// timing.cu — per-launch device timing by kernel category (timing.h).  Process-wide state behind one mutex: arming,
// recording and reading may come from different host threads; the events are recorded on the launching stream.
#include "timing.h"

#include <mutex>
#include <vector>

#include "zkd_internal.h"

namespace zkd {

namespace {
struct Slot {
  int cat;
  uint64_t work_exec, work_alg;
};
struct State {
  std::mutex mu;
  bool enabled = false;
  std::vector<cudaEvent_t> ev;  // pairs, grow-only pool
  std::vector<Slot> slots;      // used pairs
  // results of the last read (events are only walked once per arming)
  bool summed = false;
  double ms[KC_NUM];
  uint64_t launches[KC_NUM], wexec[KC_NUM], walg[KC_NUM];
};
State& st() {
  static State s;
  return s;
}
constexpr size_t kMaxTimed = 1u << 16;
}  // namespace

const char* kcat_name(int cat) {
  switch (cat) {
    case KC_GEMM_DIGITS: return "gemm_digits_kernel";
    case KC_GEMM_I8: return "gemm_i8_kernel";
    case KC_SEED: return "seed_fp64";
    case KC_SSTEP: return "singleton_step_kernel";
    case KC_PREP: return "prep_kernel";
    case KC_COMBINE: return "combine_kernel";
    case KC_SLICE_I8: return "slice_i8_kernel";
    case KC_COMBINE_I8: return "combine_i8_kernel";
    case KC_ECALC: return "ecalc_kernel";
    case KC_LU: return "lu_kernels";
    case KC_IO: return "ingest_export";
    case KC_OTHER: return "other";
    default: return nullptr;
  }
}

bool kt_armed() { return st().enabled; }

void kt_enable(bool on) {
  State& s = st();
  std::lock_guard<std::mutex> lk(s.mu);
  s.enabled = on;
  if (on) {
    s.slots.clear();
    s.summed = false;
  }
}

KtScope::KtScope(int cat, cudaStream_t stream, uint64_t work_exec, uint64_t work_alg) : slot_(-1), s_(stream) {
  State& s = st();
  if (!s.enabled) return;
  std::lock_guard<std::mutex> lk(s.mu);
  if (!s.enabled || s.slots.size() >= kMaxTimed) return;
  const size_t i = s.slots.size();
  while (s.ev.size() < 2 * (i + 1)) {
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) {
      (void)cudaGetLastError();
      return;
    }
    s.ev.push_back(e);
  }
  s.slots.push_back(Slot{cat, work_exec, work_alg ? work_alg : work_exec});
  s.summed = false;
  slot_ = (int)i;
  cudaEventRecord(s.ev[2 * i], stream);
}

KtScope::~KtScope() {
  if (slot_ < 0) return;
  State& s = st();
  std::lock_guard<std::mutex> lk(s.mu);
  if ((size_t)slot_ < s.slots.size()) cudaEventRecord(s.ev[2 * (size_t)slot_ + 1], s_);
}

int kt_read(int cat, double* ms, uint64_t* launches, uint64_t* work_exec, uint64_t* work_alg) {
  if (cat < 0 || cat >= KC_NUM) return ZKD_ERR_INVALID_ARG;
  State& s = st();
  std::lock_guard<std::mutex> lk(s.mu);
  if (!s.summed) {
    for (int c = 0; c < KC_NUM; ++c) { s.ms[c] = 0; s.launches[c] = 0; s.wexec[c] = 0; s.walg[c] = 0; }
    for (size_t i = 0; i < s.slots.size(); ++i) {
      float t = 0;
      if (cudaEventSynchronize(s.ev[2 * i + 1]) != cudaSuccess || cudaEventElapsedTime(&t, s.ev[2 * i], s.ev[2 * i + 1]) != cudaSuccess) {
        (void)cudaGetLastError();
        return ZKD_ERR_CUDA;
      }
      const Slot& sl = s.slots[i];
      s.ms[sl.cat] += t;
      s.launches[sl.cat] += 1;
      s.wexec[sl.cat] += sl.work_exec;
      s.walg[sl.cat] += sl.work_alg;
    }
    s.summed = true;
  }
  if (ms) *ms = s.ms[cat];
  if (launches) *launches = s.launches[cat];
  if (work_exec) *work_exec = s.wexec[cat];
  if (work_alg) *work_alg = s.walg[cat];
  return ZKD_OK;
}

}  // namespace zkd
