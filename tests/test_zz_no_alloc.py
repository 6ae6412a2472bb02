"""vd_nearest_static: the nearest-site query without any device allocation (queries and results staged in a fixed device
array inside the library, include/vd.h).  Its output must equal vd_nearest's -- the existing path, itself checked against
brute force in test_gpu_parity.py -- exactly (site ids), on two calls in a row that share the scratch array, the second one
smaller than the first so that stale contents would show.  This file is collected last on purpose."""
import numpy as np
import pytest

from paper_2509_07175_b200 import binding, inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("idx", [2, 3, 1])      # uniform 3D, clustered 3D (refined index), 2D
def test_nearest_static_equals_nearest_on_two_calls_in_a_row(idx):
    import torch
    w = inputs.config(idx, "small")
    dim = w.sites.shape[1]
    rng = np.random.default_rng(900 + idx)
    qa = np.concatenate([rng.random((5000, dim)), rng.random((600, dim)) * 4.0 - 1.5, w.sites[rng.integers(0, w.n, 300)] + 1e-7])
    qb = rng.random((1234, dim)) * 1.2 - 0.1
    with binding.Context(w.sites) as ctx:
        with pytest.raises(binding.VdError) as e:            # no index yet: building one would allocate
            ctx.nearest_static(qa)
        assert e.value.status == 3
        ref_a, ref_b = ctx.nearest(qa), ctx.nearest(qb)     # the existing path (builds the index)
        brute = ((qb[:, None, :] - w.sites[None, :, :]) ** 2).sum(-1).argmin(1)
        assert np.array_equal(ref_b, brute)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        got_a = ctx.nearest_static(qa)
        got_b = ctx.nearest_static(qb)                        # right after, into the same scratch array
        # device pointers in, device pointer out
        dq = torch.from_numpy(qa).cuda()
        dout = torch.empty(len(qa), dtype=torch.int32, device="cuda")
        free1 = torch.cuda.mem_get_info()[0]
        ctx.nearest_static(dq, out=dout)
        got_c = ctx.nearest_static(qb)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free1          # the calls took no device memory
        assert free1 <= free0
        assert np.array_equal(got_a, ref_a) and np.array_equal(got_b, ref_b)
        assert np.array_equal(dout.cpu().numpy(), ref_a) and np.array_equal(got_c, ref_b)
        # limits and errors
        with pytest.raises(binding.VdError) as e:
            ctx.nearest_static(np.zeros((65537, dim)))
        assert e.value.status == 1 and "65536" in str(e.value)
        bad = qb.copy()
        bad[7, 0] = np.nan
        with pytest.raises(binding.VdError) as e:
            ctx.nearest_static(bad)
        assert e.value.status == 4
        assert np.array_equal(ctx.nearest_static(qb), ref_b)  # the flag was cleared: the next call is clean
        assert np.array_equal(ctx.nearest_static(np.ascontiguousarray(qa[:65536 if len(qa) > 65536 else len(qa)])), ref_a)
