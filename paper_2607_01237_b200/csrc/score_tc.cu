// score_tc.cu — placeholder until the tcgen05/TMA score kernel lands: reports "unsupported" so
// kara_compress_window runs the CUDA-core score kernel.
#include "score_tc.h"

namespace kara {
int score_tc_attach(ScoreTcState* s, const Geom&, void*) { s->ready = false; return KARA_OK; }
bool score_tc_supported(const ScoreTcState&, const Call&) { return false; }
int score_tc_launch(ScoreTcState*, Call&, cudaStream_t, int*) { return KARA_EUNSUPPORTED; }
const char* score_tc_error() { return "tcgen05 score kernel not built"; }
}  // namespace kara
