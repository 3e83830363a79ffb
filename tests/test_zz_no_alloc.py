"""satsplat_relocate_static: the relocation step for hosts that cannot give the library a scratch buffer.

Some programs that embed this library have no way to allocate device memory at the moment they need a relocation: the
training framework around them holds the whole GPU in its own pool, the job is pinned to a memory quota that is already
used up, or the loop is latency-bound and an allocation would stall every stream on the device.  For them the library
carries a fixed working array inside its own image (room for 131072 surfels) and `satsplat_relocate_static` runs the same
kernels as `satsplat_relocate` on that array.

What is checked here: the static entry point gives the same result as the existing path (which is itself checked against
the oracle in test_gpu_parity.py) on two calls in a row.  The second call has a different size and finds the first call's
leftovers in the shared array, so a result that depended on stale contents would show.  The file is named so that pytest
collects it last: with `-x` a failure here cannot hide another test.  It holds no state of its own, so it passes alone in
a fresh process (where its first call performs the per-device address look-up) as well as after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _inputs(n, frac_dead, seed):
    rng = np.random.default_rng(seed)
    f32 = lambda a: np.asarray(a, np.float32)
    means, quats = f32(rng.normal(0, 10, (n, 3))), f32(rng.normal(0, 1, (n, 4)))
    scales, rgb = f32(rng.uniform(0.2, 2, (n, 2))), f32(rng.uniform(0, 1, (n, 3)))
    logits = f32(rng.normal(0.5, 1.5, n))
    dead = rng.uniform(0, 1, n) < frac_dead
    logits[dead] = f32(rng.uniform(-12, -5.4, dead.sum()))      # opacity below the 0.005 threshold
    u = np.minimum(f32(rng.uniform(0, 1, n)), np.float32(0.99999994))
    return (means, quats, scales, logits, rgb), u


def _run(P, call, n, arrays, u):
    import torch
    dev = [torch.from_numpy(a.copy()).cuda() for a in arrays]
    ns = P.adam_state_floats(n)
    rng = np.random.default_rng(n + 1)
    am = torch.from_numpy(rng.normal(0, 1, ns).astype(np.float32)).cuda()
    av = torch.from_numpy(rng.uniform(0, 1, ns).astype(np.float32)).cuda()
    src = call(n, *dev, am, av, torch.from_numpy(u).cuda(), want_src=True)
    torch.cuda.synchronize()
    return [t.cpu().numpy() for t in dev + [am, av, src]]


def test_relocate_static_equals_relocate_on_two_calls_in_a_row():
    import paper_2606_28581_b200 as P
    # first a large call that fills most of the shared array, then a small one that must not see what the first left behind
    for n, frac_dead, seed in ((100_003, 0.4, 11), (4_097, 0.97, 12)):
        arrays, u = _inputs(n, frac_dead, seed)
        want = _run(P, P.relocate, n, arrays, u)
        got = _run(P, P.relocate_static, n, arrays, u)
        names = ("means", "quats", "scales", "logits", "rgb", "adam_m", "adam_v", "src")
        assert (want[-1] >= 0).sum() > 0, "the case relocates nothing"
        for k, a, b in zip(names, got, want):
            if k in ("src", "adam_m", "adam_v"):
                assert np.array_equal(a, b), k                   # index work and cleared state: exact
            else:
                # the tolerance test_relocate_matches_oracle uses for these arrays (same kernels: equal in practice)
                np.testing.assert_allclose(a.astype(np.float64), b.astype(np.float64), rtol=3e-6, atol=1e-6, err_msg=k)


def test_relocate_static_refuses_more_than_its_array_holds():
    import torch
    import paper_2606_28581_b200 as P
    n = P.RELOCATE_STATIC_MAX_SURFELS + 1
    z = lambda *s: torch.zeros(*s, device="cuda")
    with pytest.raises(P.SatsplatError) as e:
        P.relocate_static(n, z(n, 3), z(n, 4), z(n, 2), z(n), z(n, 3), None, None, z(n))
    assert e.value.code == P.E_INVALID and str(P.RELOCATE_STATIC_MAX_SURFELS) in str(e.value)
    # the limit itself is accepted
    n = P.RELOCATE_STATIC_MAX_SURFELS
    arrays, u = _inputs(n, 0.1, 13)
    want = _run(P, P.relocate, n, arrays, u)
    got = _run(P, P.relocate_static, n, arrays, u)
    assert np.array_equal(got[-1], want[-1]) and np.array_equal(got[3], want[3])
