"""GPU parity of image_reproject (kernel K11) with the oracle O12 (oracle/reproject.py), through the C ABI.
PAPER.md:114, readings R1-R6.  Tolerance: 1e-6 * max|src| (float32 blend of float32 pixels with float32 fractions of
float64 coordinates: a few ulp of the largest neighbour; R6)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import reproject as orp  # noqa: E402
from synth import CONFIGS, make_frames  # noqa: E402


@pytest.fixture(scope="module")
def bd():
    import paper_2502_10783_b200 as m
    return m


@pytest.fixture(scope="module")
def ctx(bd):
    c = bd.Context(0)
    yield c
    c.close()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rot(th, s=1.0, sh=0.0, tx=0.0, ty=0.0):
    return [s * np.cos(th), -s * np.sin(th) + sh, tx, s * np.sin(th), s * np.cos(th), ty]


@pytest.mark.parametrize("Hs,Ws,out_shape,fill", [(97, 132, None, 0.0), (64, 64, (80, 96), -3.5), (300, 260, (130, 516), 7.0), (5, 8, (9, 12), 1.0)])
def test_k11_every_pixel(bd, ctx, Hs, Ws, out_shape, fill):
    rng = np.random.default_rng(Hs + Ws)
    mats = [rot(0.0), rot(0.0, tx=3.0, ty=-2.0), rot(0.2, 1.0, 0.0, 2.3, -1.7), rot(-0.7, 0.9, 0.15, 10.0, 6.5), rot(2.5, 1.3, -0.2, 0.6 * Ws, 0.5 * Hs),
            rot(0.001, 1.0005, 0.0, -0.37, 0.81), [1, 2, 0, 2, 4, 0], rot(0.3, 40.0), rot(0.3, 0.02, 0.0, 0.4 * Ws, 0.4 * Hs), [1, 0, 1e300, 0, 1, 0],
            rot(-0.003, 0.9995, 0.0, 1.25, 2.5), [1, 0, 0.3, 0.01, 1, -0.2], [1, 0, -0.6, -0.02, 1.0, 0.7], rot(0.004, 1.0007, 0.0006, 3.37, -2.81)]
    B = len(mats)
    src = rng.normal(1000, 200, size=(B, Hs, Ws)).astype(np.float32)
    out = bd.image_reproject(ctx, dev(src), dev(np.array(mats, dtype=np.float64)), out_shape, fill)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    tol = 1e-6 * float(np.abs(src).max())
    for f, A in enumerate(mats):
        want = orp.reproject(src[f], A, out_shape, fill)
        assert got[f].shape == want.shape
        assert np.max(np.abs(got[f] - want)) <= tol, (f, np.max(np.abs(got[f] - want)))
    # identity and integer shifts reproduce source pixels bit for bit (weights 0 and 1 are exact)
    if out_shape is None:
        assert np.array_equal(got[0], src[0])
        assert np.array_equal(got[1][:-2, 3:], src[1][2:, :-3]) and np.all(got[1][-2:, :] == np.float32(fill))
    assert np.all(got[6] == np.float32(fill))       # R5: singular
    # deterministic
    out2 = bd.image_reproject(ctx, dev(src), dev(np.array(mats, dtype=np.float64)), out_shape, fill)
    assert torch.equal(out, out2)


def test_k11_rejects_bad_arguments(bd, ctx):
    src = torch.zeros((1, 16, 16), dtype=torch.float32, device="cuda")
    A = dev(np.array([rot(0.1)]))
    with pytest.raises(bd.BkgdetError):
        bd.image_reproject(ctx, src, A, (16, 18))            # result width not a multiple of 4
    with pytest.raises(bd.BkgdetError):
        bd.image_reproject(ctx, src, dev(np.zeros((2, 6))))  # one matrix per frame
    with pytest.raises(bd.BkgdetError):
        bd.image_reproject(ctx, src, A, out=src)             # in place


def test_k11_full_size_config3(bd, ctx):
    """The launch configuration bench.py times (9216 x 9232, a rotation + shear + shift of survey size): sampled result pixels
    (random, the four corners, the rim where the border is interpolated) against the oracle, one by one."""
    cfg = CONFIGS[3]
    img = make_frames(cfg)
    _, H, W = img.shape
    A = rot(0.004, 1.0007, 0.0006, 3.37, -2.81)
    out = bd.image_reproject(ctx, dev(img), dev(np.array([A])), None, 0.0)
    torch.cuda.synchronize()
    got = out[0].cpu().numpy()
    rng = np.random.default_rng(12)
    ys = np.concatenate([rng.integers(0, H, 40000), [0, 0, H - 1, H - 1], rng.integers(0, 45, 2000), rng.integers(H - 45, H, 2000)])
    xs = np.concatenate([rng.integers(0, W, 40000), [0, W - 1, 0, W - 1], rng.integers(0, W, 2000), rng.integers(0, W, 2000)])
    want = orp.reproject(img[0], A, None, 0.0, only=(ys, xs))
    tol = 1e-6 * float(np.abs(img).max())
    assert np.max(np.abs(got[ys, xs] - want)) <= tol
    inv = orp.invert_affine(A)
    for y, x in zip(ys[:200], xs[:200]):
        assert abs(got[y, x] - orp.reproject_pixel(img[0], inv, int(x), int(y), 0.0)) <= tol
    # the result is not the source (the map is not the identity) and holds fill where the source does not reach
    assert not np.array_equal(got, img[0]) and (got == 0.0).any()
