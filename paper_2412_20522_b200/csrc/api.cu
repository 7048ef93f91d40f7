// api.cu -- error reporting and version of libmg.
#include <cstdarg>
#include <cstdio>

#include "mg_common.cuh"

static thread_local char g_err[512] = "";

void mg_set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

int mg_current_device(int* dev, int* sm_count) {
  static int sms_of[64];  // 0 = not asked yet; written atomically, the value is the same whoever writes it
  int d = 0;
  MG_CHECK_CUDA(cudaGetDevice(&d));
  int sms = __atomic_load_n(&sms_of[d & 63], __ATOMIC_ACQUIRE);
  if (sms == 0 || d >= 64) {
    MG_CHECK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, d));
    if (d < 64) __atomic_store_n(&sms_of[d], sms, __ATOMIC_RELEASE);
  }
  if (dev) *dev = d;
  if (sm_count) *sm_count = sms;
  return MG_OK;
}

extern "C" const char* mg_last_error_string(void) { return g_err; }
extern "C" int mg_version(void) { return 200; }
