"""ks_predict_routed_static (include/ks.h): density-routed prediction whose scratch (the row lists of the routing
pass) lives in a fixed device array of libks instead of the context's cudaMalloc'ed workspace.

Checked against the existing path, ks_predict_kernels(KS_TIER_B_ROUTED, KS_MEM_DEVICE), on the same device buffers:
the same kernels run, so tiles/waves must be equal and latencies agree within the fp32 tolerance of the parity
tests (they are in fact bit-equal: the order of a row list varies, the results do not).  Collected last on purpose
(the suite runs with pytest -x): the file name sorts after every other test file."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL_F32 = 1e-5     # tests/test_gpu_parity.py: the fp32 paths


def rel_err(got, want):
    want = np.asarray(want, np.float64)
    return np.abs(np.asarray(got, np.float64) - want) / np.maximum(np.abs(want), 1e-300)


@pytest.fixture(scope="module")
def ks():
    import torch
    from paper_2606_28565_b200 import binding as B
    from paper_2606_28565_b200 import build as ksbuild
    from paper_2606_28565_b200 import driver as D
    ksbuild.build()
    assert torch.cuda.is_available()
    return B, D


def outputs(torch, db, ns, fill=None):
    mk = (lambda dt: [torch.empty((ns, b.n), dtype=dt, device="cuda:0") for b in db]) if fill is None else \
         (lambda dt: [torch.full((ns, b.n), fill, dtype=dt, device="cuda:0") for b in db])
    return mk(torch.float32), mk(torch.int32), mk(torch.int32), mk(torch.float32)


def routed_workload(n, n_specs):
    w = W.config3(n=n, routed=True)
    w.specs = [W.spec_gb200(), W.spec_gb200(n_sm=132, peak_flops=1.0e15, peak_bw=3.35e12, t0=3e-6),
               W.spec_gb200(ctas_per_sm=2)][:n_specs]
    return w


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row(ks):
    B, D = ks
    import torch
    # two workloads of different sizes: the second call finds the first call's lists in the array
    cases = [routed_workload(30011, 3), routed_workload(5003, 1)]
    ctx_ref, ctx = B.Context(0), B.Context(0)     # ctx never owns a workspace: nothing but its models is allocated
    try:
        for round_ in range(2):
            for w in cases:
                D.load_models(ctx_ref, w)
                D.load_models(ctx, w)
                db = D.to_device(w)
                ns = len(w.specs)
                ref = outputs(torch, db, ns)
                got = outputs(torch, db, ns)
                ctx_ref.predict_kernels(db, w.specs, W.TIER_B_ROUTED, *ref, space=B.KS_MEM_DEVICE)
                torch.cuda.synchronize()
                free0 = torch.cuda.mem_get_info(0)[0]
                ctx.predict_routed_static(db, w.specs, *got)
                ctx.predict_routed_static(db, w.specs, *got)          # back to back on one stream: ordered, no race
                torch.cuda.synchronize()
                free1 = torch.cuda.mem_get_info(0)[0]
                if round_ == 1:                                        # every kernel has run once: the device's free
                    assert free1 >= free0                              # memory does not shrink across the calls
                routed_any = False
                for i, b in enumerate(db):
                    lat_r, lat_g = ref[0][i].cpu().numpy(), got[0][i].cpu().numpy()
                    assert np.array_equal(ref[1][i].cpu().numpy(), got[1][i].cpu().numpy())      # tiles
                    assert np.array_equal(ref[2][i].cpu().numpy(), got[2][i].cpu().numpy())      # waves
                    assert rel_err(got[3][i].cpu().numpy(), ref[3][i].cpu().numpy()).max(initial=0) <= TOL_F32
                    assert np.isfinite(lat_g).all() and (lat_g > 0).all()
                    assert rel_err(lat_g, lat_r).max(initial=0) <= TOL_F32
                    assert np.array_equal(lat_g, lat_r)
                    # the routing pass did something: Tier B alone differs on the rows outside the hull
                    tb = torch.empty((ns, b.n), dtype=torch.float32, device="cuda:0")
                    ctx_ref.predict_kernels([b], w.specs, W.TIER_B, [tb], space=B.KS_MEM_DEVICE)
                    torch.cuda.synchronize()
                    routed_any |= bool((tb.cpu().numpy() != lat_g).any())
                assert routed_any
    finally:
        ctx.close()
        ctx_ref.close()


def test_static_scratch_rejects_sizes_beyond_its_maximum(ks):
    B, D = ks
    import torch
    w = routed_workload(4001, 1)
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        gemm = next(b for b in w.buckets if b.family == W.FAM_GEMM)
        n_big = B.KS_STATIC_ROUTE_MAX_ROWS + 4
        reps = -(-n_big // gemm.n)

        class Big:
            family, dtype_bytes, hq, hkv, head_dim = gemm.family, gemm.dtype_bytes, gemm.hq, gemm.hkv, gemm.head_dim
            model_slot, mult = gemm.model_slot, None
            cols = [torch.from_numpy(np.tile(np.asarray(c), reps)[:n_big].copy()).to("cuda:0") for c in gemm.cols]
            n = n_big

        lat = [torch.full((1, n_big), -1.0, dtype=torch.float32, device="cuda:0")]
        with pytest.raises(B.KsError) as ei:
            ctx.predict_routed_static([Big], w.specs, lat)
        assert ei.value.status == B.KS_ELIMIT and "KS_ELIMIT" in str(ei.value)
        torch.cuda.synchronize()
        assert bool((lat[0] == -1.0).all())                           # nothing was enqueued or written
        # exactly at the maximum it runs, and agrees with the workspace path
        n_max = B.KS_STATIC_ROUTE_MAX_ROWS

        class Max(Big):
            cols = [c[:n_max].contiguous() for c in Big.cols]
            n = n_max

        got = [torch.empty((1, n_max), dtype=torch.float32, device="cuda:0")]
        ref = [torch.empty((1, n_max), dtype=torch.float32, device="cuda:0")]
        ctx.predict_routed_static([Max], w.specs, got)
        ctx.predict_kernels([Max], w.specs, W.TIER_B_ROUTED, ref, space=B.KS_MEM_DEVICE)
        torch.cuda.synchronize()
        assert rel_err(got[0].cpu().numpy(), ref[0].cpu().numpy()).max() <= TOL_F32
    finally:
        ctx.close()
