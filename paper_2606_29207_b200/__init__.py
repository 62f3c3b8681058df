"""paper_2606_29207_b200 -- B200-native hot path of KernelFlume (arxiv/paper_2606_29207):
split-KV GQA decode attention over token-range KV partitions + LSE merge + KV append / route update,
as hand-written CUDA for sm_100a behind a C ABI (include/kflume.h, csrc/)."""
from .binding import (KF_ECUDA, KF_EINVAL, KF_ENOSPC, KF_ESTATE, KF_IMPL_AUTO, KF_IMPL_SIMPLE, KF_IMPL_TMA,  # noqa: F401
                      KF_OK, KF_W_DOWN, KF_W_GATE, KF_W_KV, KF_W_O, KF_W_Q, KF_W_UP, KFlume, KFlumeError, Policy, StepGraph,
                      WSide, kf_config, kf_policy_config, kf_wside_config, load_library, make_config)
