"""kf_attend_static: the attend + merge launch for callers that can neither pass scratch memory nor allocate it.

Who needs it: an attention node that has handed every byte of its HBM to KV pools and is then pulled into a running
decode loop, a thread that must keep out of the CUDA allocator because cudaMalloc / cudaFree synchronise the whole
device (and would stall step graphs replaying on other streams), or code under a framework whose own caching allocator
owns all device memory.  For them the range partials live in a fixed array inside the library image
(KF_STATIC_SCRATCH_BYTES per GPU, held until the process exits) -- see include/kflume.h.

What is checked: on two decode steps in a row the new entry point returns what the existing kf_attend returns (the
same kernel, plan and merge order: bit for bit, hence also inside the suite's tolerance) and what the fp64 oracle
says.  The second call finds the array full of the first call's partials (other lengths, other q), so a kernel that
read anything it had not written itself would show up here.  A config whose partials exceed the array is refused with
KF_EINVAL and a message that names the sizes.

This file sorts last on purpose (pytest -x stops at the first failure; nothing is hidden behind this one), and it
passes alone in a fresh process as well as after the rest of the suite: the first call on a GPU looks the array's
address up, whoever makes it.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from kf_inputs.workloads import Workload  # noqa: E402
from kf_testlib import LSE_REL_TOL, O_ABS_TOL, check_close, oracle_request  # noqa: E402
from paper_2606_29207_b200 import KF_EINVAL, KF_OK, KFlume, KFlumeError, make_config  # noqa: E402
from paper_2606_29207_b200.binding import load_library  # noqa: E402
from paper_2606_29207_b200.workload import Session  # noqa: E402

STATIC_BYTES = 16 << 20   # KF_STATIC_SCRATCH_BYTES of include/kflume.h


def test_static_scratch_matches_existing_path_on_two_calls_in_a_row():
    # ragged contexts over several 64-token ranges on 3 partitions: 1, 2, 4, 9 and 4 ranges, so the launch merges
    # pieces -> range partials -> outputs through the scratch; request 1 fills its range after step 0 and opens a new one
    wl = Workload("no_alloc", 32, 8, 64, 3, [33, 128, 200, 515, 256], n_steps=2)
    ses = Session(wl)
    ses.prepare()
    kf = ses.kf
    o_a, lse_a = torch.empty_like(ses.o), torch.empty_like(ses.lse)
    for step in range(2):
        kf.token_boundary()
        q = ses.q_for(0, step)
        k_new, v_new = ses.kv_new_for(0, step)
        kf.kv_append(0, k_new, v_new)
        # the existing path (partials in the ctx workspace), then the entry point under test on the same state;
        # outputs are pre-filled with NaN so that a row left unwritten cannot pass
        ses.o.fill_(float("nan")), ses.lse.fill_(float("nan"))
        o_a.fill_(float("nan")), lse_a.fill_(float("nan"))
        kf.attend(0, q, ses.o, ses.lse)
        kf.attend_static(0, q, o_a, lse_a)
        kf.step_commit()
        assert kf.status() == KF_OK
        o_ref, lse_ref = ses.o.cpu().numpy(), ses.lse.cpu().numpy()
        o_new, lse_new = o_a.cpu().numpy(), lse_a.cpu().numpy()
        assert np.isfinite(o_new).all() and np.isfinite(lse_new).all(), f"step {step}: unwritten or non-finite rows"
        # within the tolerance the parity tests use (north_star: 2e-3 on o, 1e-4 relative on lse) ...
        assert np.abs(o_new - o_ref).max() <= O_ABS_TOL, f"step {step}"
        assert (np.abs(lse_new - lse_ref) <= LSE_REL_TOL * np.maximum(1.0, np.abs(lse_ref))).all(), f"step {step}"
        # ... and in fact identical: only the address of the partials differs between the two launches
        assert np.array_equal(o_new.view(np.uint32), o_ref.view(np.uint32)), f"step {step}: o differs from kf_attend"
        assert np.array_equal(lse_new.view(np.uint32), lse_ref.view(np.uint32)), f"step {step}: lse differs from kf_attend"
        # and against the oracle, so that "equal" cannot mean "equally wrong"
        for r, S0 in enumerate(wl.contexts):
            o_star, lse_star = oracle_request(wl, 0, r, step, S0 + step)
            check_close(o_new[r], lse_new[r], o_star, lse_star, f"static scratch, step {step}, request {r}")
    assert kf.route_snapshot()["n_ranges"] == [1, 3, 4, 9, 5]
    ses.close()


def test_static_scratch_rejects_a_config_beyond_its_size():
    # B * Jmax * H_q * (128 + 1) * 4 bytes: 64 * 32 * 32 * 516 = 33.8 MB > 16 MiB; nothing is launched
    B, Jmax, Hq = 64, 32, 32
    assert B * Jmax * Hq * 129 * 4 > STATIC_BYTES
    kf = KFlume(make_config(Hq, 8, 16, 2, B, Jmax, 8))
    q = torch.zeros((B, Hq, 128), dtype=torch.float16, device=kf.device)
    o = torch.zeros((B, Hq, 128), dtype=torch.float32, device=kf.device)
    lse = torch.zeros((B, Hq), dtype=torch.float32, device=kf.device)
    before = kf.launch_count()
    with pytest.raises(KFlumeError) as err:
        kf.attend_static(0, q, o, lse)
    assert err.value.code == KF_EINVAL
    assert "KF_STATIC_SCRATCH_BYTES" in str(err.value) and str(B * Jmax * Hq) in str(err.value)
    assert kf.launch_count() == before
    # the largest shape that still fits is accepted: 16 MiB / (129 * 4 B) rows, less the alignment padding
    kf.close()
    B2, Jmax2 = 32, 31     # 32 * 31 * 32 rows * 516 B = 16.38e6 <= 16 MiB
    assert (B2 * Jmax2 * Hq * 512 + 255) // 256 * 256 + B2 * Jmax2 * Hq * 4 <= STATIC_BYTES
    kf = KFlume(make_config(Hq, 8, 16, 2, B2, Jmax2, 8))
    q = torch.zeros((B2, Hq, 128), dtype=torch.float16, device=kf.device)
    o = torch.zeros((B2, Hq, 128), dtype=torch.float32, device=kf.device)
    lse = torch.zeros((B2, Hq), dtype=torch.float32, device=kf.device)
    kf.token_boundary()
    kf.attend_static(0, q, o, lse)     # no open request: a launch with nothing to do
    assert kf.status() == KF_OK
    kf.close()
    assert load_library().kf_attend_static(None, 0, None, None, None, None) == KF_EINVAL
