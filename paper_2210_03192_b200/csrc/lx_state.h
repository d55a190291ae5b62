// lx_state.h — the few pieces of library state (lx_api.cu) other translation units need.
#pragma once
namespace lx {
bool state_ready();
const double *state_boys_tab();
int state_num_sms();
void state_count_launches(int n);
int state_cuda_fail(int cuda_error);   // records the message for lx_strerror, returns LX_ECUDA
}  // namespace lx
