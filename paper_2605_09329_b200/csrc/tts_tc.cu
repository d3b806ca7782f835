// placeholder: tensor-core path not built yet
#include "tts_internal.h"
namespace tts {
bool tc_supported(const tts_config&) { return false; }
cudaError_t tc_init(tts_ctx*) { return cudaSuccess; }
void tc_destroy(tts_ctx*) {}
cudaError_t tc_step(tts_ctx*, const StepArgs&, cudaStream_t, int*) { return cudaErrorNotSupported; }
}  // namespace tts
