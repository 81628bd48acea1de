#include "ozfft.h"
extern "C" {
ozfft_plan ozfft_plan_create(int, int, int, int) { return nullptr; }
ozfft_plan ozfft_plan_create_1d(int, int, int) { return nullptr; }
int ozfft_exec(ozfft_plan, const void *, void *, void *) { return OZFFT_EINVAL; }
int ozfft_exec_host(ozfft_plan, const void *, void *, void *) { return OZFFT_EINVAL; }
void ozfft_plan_destroy(ozfft_plan) {}
const char *ozfft_last_error(void) { return "stub"; }
uint64_t ozfft_twiddle_checksum(void) { return 0; }
int ozfft_plan_num_launches(ozfft_plan) { return 0; }
size_t ozfft_plan_device_bytes(ozfft_plan) { return 0; }
int ozfft_exec_axis(ozfft_plan, int, const void *, void *, void *) { return OZFFT_EINVAL; }
}
