"""GPU checks of the C-ABI's call rules (include/apic.h), as opposed to its arithmetic: what happens when the
families of entries are mixed on one plan, and that plan-time limits are reported as parameter errors."""
import numpy as np
import pytest

from apic_synth import get_config, make_batch
from helpers import plan_from_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def A():
    import torch
    assert torch.cuda.is_available()
    import paper_2407_20469_b200 as pkg
    pkg.load()
    return pkg


def test_device_entry_issued_while_a_submitted_batch_is_in_flight(A):
    """apic_submit_host(slot 0) and apic_reconstruct share workspace set 0.  The device entry must first complete the
    batch in flight (apic.h, "Mixing with the device-pointer entries"), so both come out with the bits they have when
    run one at a time, whichever order and however often the two are interleaved; the same for the stage buffers
    read through apic_debug_copy."""
    import torch
    cfg = get_config(2, tile_n=64, batch=4, grid=(2, 2))
    stacks, _ = make_batch(cfg, [0, 1, 2, 3])
    plan = plan_from_config(A, cfg, max_batch=12)
    big = np.ascontiguousarray(np.concatenate([stacks] * 3))               # 12 tiles: the batch in flight
    small = np.ascontiguousarray(stacks[::-1])                             # 4 other tiles: the device-pointer call
    d_small = torch.from_numpy(small).cuda()
    ref_big = [o.cpu().numpy() for o in plan.reconstruct(torch.from_numpy(big).cuda())]
    ref_small = [o.cpu().numpy() for o in plan.reconstruct(d_small)]
    og_small = plan.debug_buffer(A.DBG_OBJECT_SPECTRUM, 4).cpu().numpy()
    torch.cuda.synchronize()
    nz, n, on = plan.nz, plan.n, plan.out_n
    x = torch.from_numpy(big).pin_memory()
    for rep in range(4):
        out = (torch.zeros((12, on, on), dtype=torch.complex64).pin_memory(), torch.zeros((12, nz), dtype=torch.float32).pin_memory(),
               torch.zeros((12, n, n), dtype=torch.complex64).pin_memory(), torch.full((12,), -1, dtype=torch.int32).pin_memory())
        plan.submit_host(0, x, *out)
        if rep == 3:
            plan.submit_host(1, x, *out)                                  # and one in the other slot (same results)
        got = plan.reconstruct(d_small)                                    # no wait_host in between
        # the submitted batch is complete as soon as the device entry has returned
        assert np.array_equal(out[0].numpy(), ref_big[0]) and np.array_equal(out[3].numpy(), ref_big[3])
        og = plan.debug_buffer(A.DBG_OBJECT_SPECTRUM, 4)
        torch.cuda.synchronize()
        plan.wait_host(0)                                                  # returns at once
        plan.wait_host(1)
        for g, r in zip(got, ref_small):
            assert np.array_equal(g.cpu().numpy(), r)
        assert np.array_equal(og.cpu().numpy(), og_small)
        for o, r in zip(out, ref_big):
            assert np.array_equal(o.numpy(), r)
    # debug copy directly after a submit: the stage buffer read is the submitted batch's last chunk, not a torn one
    plan.submit_host(0, x, *out)
    og = plan.debug_buffer(A.DBG_OBJECT_SPECTRUM, 4)
    torch.cuda.synchronize()
    plan.wait_host(0)
    plan.reconstruct(torch.from_numpy(big).cuda())
    og_ref = plan.debug_buffer(A.DBG_OBJECT_SPECTRUM, 4)
    torch.cuda.synchronize()
    assert np.array_equal(og.cpu().numpy(), og_ref.cpu().numpy())
