/* literal.cu -- placeholder until the literal P x P chain lands (next commit). */
#include "internal.h"
int shwfs_literal_supported(const shwfs_handle *) { return 0; }
cudaError_t shwfs_literal_build_khat(shwfs_handle *, cudaStream_t) { return cudaErrorNotSupported; }
cudaError_t shwfs_literal_launch(shwfs_handle *, const float *, int, float *, int, float *, cudaStream_t) { return cudaErrorNotSupported; }
