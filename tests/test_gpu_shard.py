"""One image shared by several GPUs: gray2_init_null_shard deals the
rays out in tiles.  The box has one GPU, so the ranks are run one after the other on it -- they are independent
by construction (no rank waits for another) -- and the gathered result must equal the undivided run bit for bit."""
import numpy as np
import pytest
import torch

from gpu_helpers import INF, image_sc, run_gpu_image
from paper_1706_07062_b200 import gray2, inputs, multi

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("prec", [gray2.F64, gray2.F32], ids=["f64", "f32"])
@pytest.mark.parametrize("world,tile", [(3, 1000), (2, 4096), (8, 257), (4, 1 << 20)])
def test_sharded_image_equals_the_undivided_image(prec, world, tile):
    cfg = inputs.CFG3_NULL.scaled(131, 77)            # 10087 rays: ragged last tile in every case
    f0, full, fstats = run_gpu_image(cfg, prec=prec)
    q = torch.empty_like(full.q)
    lam, status, nsteps = torch.empty_like(full.lam), torch.empty_like(full.status), torch.empty_like(full.nsteps)
    steps = 0
    for rank in range(world):
        idx = multi.shard_global_index(cfg.n, tile, rank, world).cuda()
        assert gray2.shard_count(cfg.n, tile, rank, world) == idx.numel()
        if idx.numel() == 0:
            with pytest.raises(gray2.Gray2Error):           # a rank without rays has nothing to initialise
                gray2.init_null_shard(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, tile, rank, world,
                                      prec=prec, out=gray2.State.empty(1, prec))
            continue
        st = gray2.init_null_shard(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, tile, rank, world, prec=prec)
        assert torch.equal(st.q, f0.q[:, idx])              # the very initial data of those rays
        assert (st.a_eff, st.kind, st.reversed, st.coords) == (f0.a_eff, f0.kind, f0.reversed, f0.coords)
        stats = gray2.new_stats()
        gray2.integrate(st, INF, image_sc(cfg)[0], stats=stats)
        steps += gray2.stats_dict(stats)["steps"]
        # what multi.gather_image does across processes, here within one
        q[:, idx], lam[idx], status[idx], nsteps[idx] = st.q, st.lam, st.status, st.nsteps
    assert steps == fstats["steps"]
    assert torch.equal(q, full.q) and torch.equal(lam, full.lam)
    assert torch.equal(status, full.status) and torch.equal(nsteps, full.nsteps)


def test_shard_argument_checks_and_single_process_gather():
    cfg = inputs.CFG1_NULL
    with pytest.raises(gray2.Gray2Error) as e:
        gray2.init_null_shard(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, 512, 2, 2)
    assert e.value.code == gray2.EINVAL
    with pytest.raises(gray2.Gray2Error):
        gray2.init_null_shard(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, 0, 0, 2)
    with pytest.raises(gray2.Gray2Error):                  # wrong size of the state
        gray2.init_null_shard(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, 512, 0, 2,
                              out=gray2.State.empty(cfg.n, gray2.F64))
    whole = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    one = gray2.init_null_shard(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, 300, 0, 1)
    assert torch.equal(one.q, whole.q)                     # a single rank owns every tile, in order
    assert torch.equal(multi.gather_image(one.q, cfg.n, 300, world=1), whole.q)
