// score_tc.h — interface of the tcgen05/TMA score kernel (a1, Eq. 4) to kara_api.cu.
#pragma once
#include "kara_internal.h"

namespace kara {

struct ScoreTcState {
  bool ready = false;
  alignas(64) unsigned char k_map[128];   // CUtensorMap of the K pool (opaque here)
  alignas(64) unsigned char q_map[128];   // CUtensorMap of window_q, rebuilt when its key changes
  const void* q_ptr = nullptr;
  long long q_key[6] = {0, 0, 0, 0, 0, 0};
  int num_sms = 0;
};

// Builds the K-pool tensor map.  Returns KARA_OK / KARA_E*; score_tc_error() has the message.
int score_tc_attach(ScoreTcState* s, const Geom& g, void* k_pool);
// True if the tcgen05 kernel takes this call's shapes (else the SIMT kernel runs).
bool score_tc_supported(const ScoreTcState& s, const Call& c);
// nullptr if the tcgen05 kernel takes the call, else why not (kara_last_score_path_reason)
const char* score_tc_unsupported_reason(const ScoreTcState& s, const Call& c);
// Launches the kernel(s); sets c.parts to the number of partial column-sum strips it writes.
int score_tc_launch(ScoreTcState* s, Call& c, cudaStream_t st, int* n_launches);
const char* score_tc_error();

}  // namespace kara
