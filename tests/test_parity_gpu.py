"""Parity of the CUDA path (through the C ABI) against the CPU oracle on identical seeded inputs.

Bar (BASELINE.json north_star; reading A13): per channel,
    max_{a1..a4, r} |F_gpu - F_oracle|  <=  1e-10 * max_{a1..a4, r} |F_oracle|.
"""
import numpy as np
import pytest

from paper_1604_07983_b200 import synth

pytestmark = pytest.mark.gpu

RTOL = 1e-10


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests need a B200")
    return torch


@pytest.fixture(scope="module")
def nbs():
    from paper_1604_07983_b200 import nbs as m
    return m


def props(L, seed=21, t=0, masses=(0.20, 0.21, 0.30), same=()):
    S = {f: synth.propagator(seed, i, t, L, masses[i]) for i, f in enumerate("uds")}
    for a, b in same:
        S[a] = S[b]
    return S


def to_dev(torch, S):
    cache = {}
    out = {}
    for f in "uds":
        key = id(S[f])
        if key not in cache:
            cache[key] = torch.from_numpy(S[f]).cuda()
        out[f] = cache[key]
    return out


def assert_parity(F_gpu, F_or, chans, scale=None):
    F_gpu = np.asarray(F_gpu)
    assert F_gpu.shape == F_or.shape
    for i, ch in enumerate(chans):
        ref = np.abs(F_or[i]).max() if scale is None else scale
        assert ref > 0
        err = np.abs(F_gpu[i] - F_or[i]).max() / ref
        assert err <= RTOL, (i, ch, err)


def run_gpu(torch, nbs, L, S, chans=None, t=0, T=1):
    with nbs.Nbs(L, T, chans) as ctx:
        d = to_dev(torch, S)
        ctx.load(t, d["u"], d["d"], d["s"])
        F = ctx.correlator(t)
        torch.cuda.synchronize()
        return F.cpu().numpy()


# ------------------------------------------------------------------------------ row a1: blocks
@pytest.mark.parametrize("L", [2, 3])
def test_normal_blocks_match_oracle(torch_cuda, nbs, oracle, L):
    """eq. 2.5 / 4.1 for all eleven interpolating fields, u != d != s."""
    S = props(L, seed=5)
    with nbs.Nbs(L, 1, [("p", "n", "p", "n")]) as ctx:
        d = to_dev(torch_cuda, S)
        ctx.load(0, d["u"], d["d"], d["s"])
        for name in oracle.BARYONS:
            got = ctx.blocks_x(0, name).cpu().numpy()
            ref = oracle.block(S, name)
            assert np.abs(got - ref).max() <= RTOL * np.abs(ref).max(), name


# ------------------------------------------------------------------------------ rows a2, a5: FFT
@pytest.mark.parametrize("L", [2, 4, 5, 6, 8, 12, 16, 24, 32, 48, 96])
def test_fft3d_matches_numpy(torch_cuda, nbs, L):
    """B~(q) = sum_x B(x) exp(-i q.x) and its inverse (eq. 2.6), ragged component count.  Powers of two: in-register
    radix 2; 6, 12, 24, 48, 96 (configs[4]): the same behind a radix-3 stage; 5: the O(L^2) transform."""
    torch = torch_cuda
    R = 37 if L < 32 else (70 if L == 48 else 5)  # 70 > 64: two component groups of the radix-3 kernel, ragged
    rng = np.random.default_rng(L)
    a = rng.standard_normal((L, L, L, R)) + 1j * rng.standard_normal((L, L, L, R))  # [z][y][x][R]
    with nbs.Nbs(L, 1, [("p", "n", "p", "n")]) as ctx:
        x = torch.from_numpy(a.reshape(L ** 3, R).copy()).cuda()
        ctx.fft3d(x)
        ref = np.fft.fftn(a, axes=(0, 1, 2)).reshape(L ** 3, R)
        assert np.abs(x.cpu().numpy() - ref).max() <= 1e-12 * np.abs(ref).max()
        ctx.fft3d(x, inverse=True)
        assert np.abs(x.cpu().numpy() - a.reshape(L ** 3, R)).max() <= 1e-13 * np.abs(a).max()


def test_fft3d_rejects_misaligned_data(torch_cuda, nbs):
    """include/nbs.h: nbs_fft3d wants 16-byte aligned data (the x-y pass copies 16 bytes at a time)."""
    torch = torch_cuda
    with nbs.Nbs(4, 1, [("p", "n", "p", "n")]) as ctx:
        buf = torch.zeros(64 * 8 * 2 + 2, dtype=torch.float64, device="cuda")
        rc = nbs.lib().nbs_fft3d(ctx.ctx, buf.data_ptr() + 8, 8, 0, None)
        assert rc == nbs.NBS_EINVAL and b"aligned" in nbs.lib().nbs_last_error(ctx.ctx)
        assert nbs.lib().nbs_fft3d(ctx.ctx, buf.data_ptr(), 8, 0, None) == 0
        torch.cuda.synchronize()


# ------------------------------------------------------------------------------ whole path
def test_config0_4cubed_NN(torch_cuda, nbs, oracle):
    """BASELINE.json configs[0]: 4^3 x 1, NN channel, u = d, seed 0.  Against tier B (all r) and
    against tier A, eq. 2.4 with the direct X-sum, at a few r."""
    cfg = synth.CONFIGS[0]
    S = synth.config_slice(cfg, 0)
    assert S["d"] is S["u"]
    ch = [("p", "n", "p", "n")]
    F = run_gpu(torch_cuda, nbs, 4, S, ch)
    B = oracle.all_blocks(S, ["p", "n"])
    assert_parity(F, oracle.correlator_fft(4, B, ch), ch)
    rs = [0, 1, 7, 63]
    Fd = oracle.correlator_direct(4, B, ch[0], rs=rs)
    assert np.abs(F[0][..., rs] - Fd[..., rs]).max() <= RTOL * np.abs(Fd).max()


def test_all_52_channels_4cubed(torch_cuda, nbs, oracle):
    """All 52 channels, non-degenerate u, d, s (the flavour structure of configs[2])."""
    S = props(4, seed=3)
    chans = oracle.channels52()
    F = run_gpu(torch_cuda, nbs, 4, S)
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    assert_parity(F, oracle.correlator_fft(4, B, chans), chans)


def test_all_52_channels_time_slice_scale(torch_cuda, nbs, oracle):
    """Late time slice: entries ~ exp(-m t), F ~ 1e-28; the bar is relative per channel (A13)."""
    S = props(2, seed=3, t=63)
    chans = oracle.channels52()
    F = run_gpu(torch_cuda, nbs, 2, S, t=63, T=64)
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    Fo = oracle.correlator_fft(2, B, chans)
    assert np.abs(Fo).max() < 1e-25
    assert_parity(F, Fo, chans)


@pytest.mark.parametrize("L", [3, 6])
def test_non_power_of_two_lattice(torch_cuda, nbs, oracle, L):
    """Ragged sizes: L = 3, 6 take the mixed-radix / generic FFT path."""
    S = props(L, seed=9, same=(("d", "u"),))
    chans = [("p", "n", "p", "n"), ("p", "L", "S0", "p"), ("L", "L", "S0", "S0"), ("Xm", "X0", "Xm", "X0")]
    F = run_gpu(torch_cuda, nbs, L, S, chans)
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    assert_parity(F, oracle.correlator_fft(L, B, chans), chans)


def test_user_channels_elementary_and_identical(torch_cuda, nbs, oracle):
    """Channels outside the 52: <p Lambda | p X_u> (eq. 2.7), pp, nn, Sigma+ Xi0."""
    S = props(2, seed=13)
    chans = [("p", "L", "p", "Xu"), ("p", "p", "p", "p"), ("n", "n", "n", "n"), ("Sp", "X0", "Sp", "X0"),
             ("Xu", "Xs", "Xd", "Xs")]
    F = run_gpu(torch_cuda, nbs, 2, S, chans)
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    assert_parity(F, oracle.correlator_fft(2, B, chans), chans)


def test_vanishing_channel_uses_pair_scale(torch_cuda, nbs, oracle):
    """u = d: the isospin-forbidden Lambda Lambda <- Sigma0 Lambda vanishes; the GPU result must be
    zero on the scale of the other channels of the same sink pair (reading A13)."""
    S = props(2, seed=4, same=(("d", "u"),))
    chans = [("L", "L", "L", "L"), ("L", "L", "S0", "L")]
    F = run_gpu(torch_cuda, nbs, 2, S, chans)
    scale = np.abs(F[0]).max()
    assert np.abs(F[1]).max() <= 1e-10 * scale


def test_channel_range_and_host_buffers(torch_cuda, nbs):
    """nbs_correlator's channel range, and host-memory input / output, give the same numbers."""
    torch = torch_cuda
    L = 4
    S = props(L, seed=8)
    full = run_gpu(torch, nbs, L, S)
    with nbs.Nbs(L, 1) as ctx:
        ctx.load(0, S["u"], S["d"], S["s"])  # numpy arrays: NBS_MEM_HOST
        part = ctx.correlator(0, 7, 19)
        host = np.empty((5, 4, 4, 4, 4, L ** 3), dtype=np.complex128)
        ctx.correlator(0, 47, 52, out=host)
        torch.cuda.synchronize()
    assert np.array_equal(part.cpu().numpy(), full[7:19])
    assert np.array_equal(host, full[47:52])


def test_two_slices_in_flight_on_two_streams(torch_cuda, nbs):
    """Row a6: slices t and t+1 pipelined on two CUDA streams equal the serial results bit for bit."""
    torch = torch_cuda
    L = 4
    chans = [("p", "n", "p", "n"), ("L", "L", "L", "L"), ("Xm", "L", "S0", "Xm")]
    Ss = [props(L, seed=30, t=t) for t in range(4)]
    serial = [run_gpu(torch, nbs, L, Ss[t], chans, t=t, T=4) for t in range(4)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    with nbs.Nbs(L, 4, chans) as ctx:
        outs = []
        devs = [to_dev(torch, S) for S in Ss]
        torch.cuda.synchronize()
        for t in range(4):
            st = streams[t % 2]
            ctx.load(t, devs[t]["u"], devs[t]["d"], devs[t]["s"], stream=st)
            outs.append(ctx.correlator(t, stream=st))
        torch.cuda.synchronize()
        for t in range(4):
            assert np.array_equal(outs[t].cpu().numpy(), serial[t]), t


def test_errors(torch_cuda, nbs):
    with pytest.raises(nbs.NbsError) as e:
        nbs.Nbs(1, 1)
    assert e.value.code == nbs.NBS_EINVAL
    with pytest.raises(nbs.NbsError) as e:
        nbs.Nbs(4, 1, [("p", "n", "p", "p")])
    assert e.value.code == nbs.NBS_EINVAL
    with nbs.Nbs(2, 2) as ctx:
        with pytest.raises(nbs.NbsError) as e:
            ctx.correlator(0)
        assert e.value.code == nbs.NBS_ESTATE
        S = to_dev(torch_cuda, props(2))
        ctx.load(0, S["u"], S["d"], S["s"])
        with pytest.raises(nbs.NbsError) as e:
            ctx.correlator(0, 5, 5)
        assert e.value.code == nbs.NBS_EINVAL
        with pytest.raises(nbs.NbsError) as e:
            ctx.correlator(0, 0, 53)
        assert e.value.code == nbs.NBS_EINVAL
        small = torch_cuda.empty(10, dtype=torch_cuda.complex128, device="cuda")
        with pytest.raises(nbs.NbsError) as e:
            ctx.correlator(0, 0, 52, out=small)
        assert e.value.code == nbs.NBS_EINVAL


def test_full_size_32cubed_52_channels_sparse_support(torch_cuda, nbs, oracle):
    """BASELINE.json configs[2] in the launch configuration bench.py times (32^3, T = 64, all 52
    channels, u != d != s), on outputs the oracle can compute one by one: the propagators of
    configs[2] are kept on 5 sites and zeroed elsewhere, so the blocks (products of propagators at
    one site) live on those sites and eq. 2.4 gives
        F(r) = sum_{(i, j): x_i - x_j = r (mod L)} pair_tensor(B1(x_i), B2(x_j)),
    non-zero at <= 21 displacements r and exactly zero at the other 32747.  The CUDA path runs its
    full-volume kernels (blocks, 32-point FFTs, product over all 32768 momenta, inverse FFT)."""
    torch = torch_cuda
    L, T, t = 32, 64, 17
    V = L ** 3
    cfg = synth.CONFIGS[2]
    sites = [(0, 0, 0), (1, 31, 5), (31, 31, 31), (16, 0, 7), (3, 30, 12)]
    idx = np.array([x + L * (y + L * z) for x, y, z in sites])
    full = synth.config_slice(cfg, t)
    S_sup = {f: np.ascontiguousarray(full[f][idx]) for f in "uds"}  # [5][12][12]
    S = {}
    for f in "uds":
        S[f] = np.zeros_like(full[f])
        S[f][idx] = S_sup[f]
    del full
    chans = oracle.channels52()
    blocks = {n: oracle.block(S_sup, n) for n in oracle.sink_names(chans)}
    ii, jj = np.meshgrid(np.arange(len(sites)), np.arange(len(sites)), indexing="ij")
    ii, jj = ii.ravel(), jj.ravel()
    rs = []
    for i, j in zip(ii, jj):
        d = [(sites[i][a] - sites[j][a]) % L for a in range(3)]
        rs.append(d[0] + L * (d[1] + L * d[2]))
    rs = np.array(rs)
    uniq = sorted(set(rs.tolist()))
    ref = np.zeros((len(chans), 256, len(uniq)), dtype=np.complex128)
    for c, ch in enumerate(chans):
        G = oracle.pair_tensor(blocks[ch[0]][ii], blocks[ch[1]][jj], ch).reshape(len(ii), 256)
        for p, r in enumerate(rs):
            ref[c, :, uniq.index(int(r))] += G[p]
    with nbs.Nbs(L, T) as ctx:
        d = to_dev(torch, S)
        ctx.load(t, d["u"], d["d"], d["s"])
        F = ctx.correlator(t).reshape(len(chans), 256, V)
        torch.cuda.synchronize()
    ref_dev = torch.from_numpy(ref).cuda()
    col = torch.tensor(uniq, device="cuda")
    scale = ref_dev.abs().amax(dim=(1, 2))
    assert float(scale.min()) > 0
    err_on = (F[:, :, col] - ref_dev).abs().amax(dim=(1, 2)) / scale
    F[:, :, col] = 0
    err_off = F.abs().amax(dim=(1, 2)) / scale
    worst = torch.maximum(err_on, err_off)
    assert float(worst.max()) <= RTOL, (int(worst.argmax()), float(err_on.max()), float(err_off.max()))


@pytest.mark.parametrize("L", [3, 4])
def test_identical_sink_baryons_only(torch_cuda, nbs, oracle, L):
    """Channel lists made of identical-baryon sinks only: the product kernel computes the momenta
    q <= -q and mirrors them to -q with the sink-swap relation (reading A11); odd L has one
    self-conjugate momentum, even L eight."""
    S = props(L, seed=17)
    chans = [("L", "L", "L", "L"), ("L", "L", "S0", "S0"), ("S0", "S0", "Sp", "Sm"), ("p", "p", "p", "p")]
    F = run_gpu(torch_cuda, nbs, L, S, chans)
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    assert_parity(F, oracle.correlator_fft(L, B, chans), chans)


def test_full_size_32cubed_isospin_relations_config3(torch_cuda, nbs):
    """BASELINE.json configs[3] (32^3, u = d = s, dense Gaussian propagators) in bench.py's launch
    configuration: the exact relations between channels of the 52-list that hold when u = d
    (pinned on the oracle in tests/test_oracle_pins.py::test_isospin_relations_u_equals_d) must hold
    on the full-volume GPU result, and the sink-swap relation for the identical-baryon sink
    Lambda Lambda (computed on half of the momenta and mirrored) must hold in r-space."""
    torch = torch_cuda
    L, T, t = 32, 64, 5
    V = L ** 3
    S = synth.config_slice(synth.CONFIGS[3], t)
    with nbs.Nbs(L, T) as ctx:
        d = to_dev(torch, S)
        ctx.load(t, d["u"], d["d"], d["s"])
        F = ctx.correlator(t).reshape(52, 4, 4, 4, 4, V)
        torch.cuda.synchronize()

    def rel(a, b):
        return float((a - b).abs().max() / torch.maximum(a.abs().max(), b.abs().max()))

    pairs = [(16, 23, +1), (17, 22, +1), (11, 12, -1), (15, 21, -1), (19, 25, -1), (20, 26, +1), (34, 35, -1),
             (38, 39, +1)]
    for i, j, sgn in pairs:
        assert rel(F[i], sgn * F[j]) <= RTOL, (i, j)
    assert rel(F[18], F[24].transpose(2, 3)) <= RTOL
    # Lambda Lambda <- Lambda Lambda (channel 10): F_{a1 a2 ..}(r) = - F_{a2 a1 ..}(-r)
    x = torch.arange(L, device="cuda")
    neg = (-x) % L
    minus_r = (neg[:, None, None] + L * (neg[None, :, None] + L * neg[None, None, :])).permute(2, 1, 0).reshape(-1)
    assert rel(F[10], -F[10].transpose(0, 1)[..., minus_r]) <= RTOL


def test_direct_shifted_sum_path(torch_cuda, nbs, oracle):
    """Row a7: eq. 2.4 as a shifted sum in x-space (nbs_set_direct), no FFT.  configs[0] (4^3, NN, u = d)
    against the oracle's direct tier A, and all 52 channels on 3^3 against tier B and the FFT path."""
    torch = torch_cuda
    S = synth.config_slice(synth.CONFIGS[0], 0)
    chans = [("p", "n", "p", "n")]
    with nbs.Nbs(4, 1, chans) as ctx:
        ctx.set_direct(True)
        d = to_dev(torch, S)
        ctx.load(0, d["u"], d["d"], d["s"])
        F = ctx.correlator(0)
        torch.cuda.synchronize()
        F = F.cpu().numpy()
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    assert_parity(F, oracle.correlator_direct(4, B, chans[0])[None], chans)

    L = 3
    S = props(L, seed=5)
    chans = oracle.channels52()
    with nbs.Nbs(L, 1) as ctx:
        d = to_dev(torch, S)
        ctx.load(0, d["u"], d["d"], d["s"])
        F_fft = ctx.correlator(0).cpu().numpy()
        ctx.set_direct(True)
        F_dir = ctx.correlator(0).cpu().numpy()
        torch.cuda.synchronize()
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    Fo = oracle.correlator_fft(L, B, chans)
    assert_parity(F_dir, Fo, chans)
    assert_parity(F_dir, F_fft, chans)
    with nbs.Nbs(16, 1, [("p", "n", "p", "n")]) as ctx, pytest.raises(nbs.NbsError):
        ctx.set_direct(True)


def test_isospin_fast_path_matches_general_path(torch_cuda, nbs, oracle):
    """with d == u (the same array) the n, Sigma-, Xi- blocks are derived from p, Sigma+, Xi0
    and neither built nor transformed.  All 52 channels against the oracle, and against the general path
    (the same values passed as two different arrays)."""
    torch = torch_cuda
    L = 4
    S = props(L, seed=12, same=(("d", "u"),))
    chans = oracle.channels52()
    F_iso = run_gpu(torch, nbs, L, S)
    with nbs.Nbs(L, 1) as ctx:
        u = torch.from_numpy(S["u"]).cuda()
        d = u.clone()  # same values, different pointer: general path
        s = torch.from_numpy(S["s"]).cuda()
        ctx.load(0, u, d, s)
        F_gen = ctx.correlator(0).cpu().numpy()
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    assert_parity(F_iso, oracle.correlator_fft(L, B, chans), chans)
    assert_parity(F_iso, F_gen, chans)


def test_isospin_channel_relations(torch_cuda, nbs, oracle):
    """VERDICT r1 item 8 / include/nbs.h nbs_set_channel_relations: with d == u nine of the 52 channels are the u <-> d
    images of earlier ones (the whole sink pair n Xi0 among them) and are written by the epilogue from their originals.
    Against the oracle and against the same run with the relations switched off, at L = 4 and at L = 6 (radix-3 FFT,
    momenta with q != -q for the mirror of the identical-baryon pairs); channel ranges that hold images without their
    originals; a user list with X fields (<n L | n Xd> = <p L | p Xu>)."""
    torch = torch_cuda
    chans = oracle.channels52()
    keep = {}
    for L, seed in ((4, 14), (6, 15)):
        S = props(L, seed=seed, same=(("d", "u"),))
        with nbs.Nbs(L, 1) as ctx:
            d = to_dev(torch, S)
            ctx.load(0, d["u"], d["d"], d["s"])
            assert ctx.derived_channels() == 9 and ctx.conjugate_pairs() == 3  # p n, Sigma+ Sigma-, Xi- Xi0
            F_rel = ctx.correlator(0).cpu().numpy()
            part = ctx.correlator(0, 21, 27).cpu().numpy()      # all of n Xi0: nothing but images
            one = ctx.correlator(0, 24, 25).cpu().numpy()       # the image with a3 <-> a4
            launches = ctx.kernel_launches()
            ctx.set_channel_relations(False)
            assert ctx.derived_channels() == 0
            F_all = ctx.correlator(0).cpu().numpy()
            ctx.set_channel_relations(True)
            assert ctx.kernel_launches() > launches
        if L == 4:
            B = oracle.all_blocks(S, oracle.sink_names(chans))
            assert_parity(F_rel, oracle.correlator_fft(L, B, chans), chans)
        assert_parity(F_rel, F_all, chans)
        assert np.array_equal(part, F_rel[21:27]) and np.array_equal(one, F_rel[24:25])
        # the relations as the oracle's pins state them (tests/test_oracle_pins.py): exact in the derived run
        assert np.array_equal(F_rel[23], F_rel[16]) and np.array_equal(F_rel[12], -F_rel[11])
        assert np.array_equal(F_rel[24], np.swapaxes(F_rel[18], 2, 3))
        keep[L] = F_rel
    # general path (d is another array): nothing is derived
    L = 4
    S = props(L, seed=14, same=(("d", "u"),))
    with nbs.Nbs(L, 1) as ctx:
        u = torch.from_numpy(S["u"]).cuda()
        ctx.load(0, u, u.clone(), torch.from_numpy(S["s"]).cuda())
        F_gen = ctx.correlator(0).cpu().numpy()
    assert_parity(keep[4], F_gen, chans)
    user = [("p", "L", "p", "Xu"), ("n", "L", "n", "Xd"), ("p", "L", "Sp", "n"), ("n", "L", "Sm", "p"), ("p", "n", "p", "n")]
    assert [r[0] for r in nbs.nbs_iso_relations(user)] == [-1, 0, -1, 2, -1]
    Fu = run_gpu(torch, nbs, L, S, user)
    B = oracle.all_blocks(S, oracle.sink_names(user))
    assert_parity(Fu, oracle.correlator_fft(L, B, user), user)
    # a list that holds channels twice: the mirror relation of the conjugate sink pairs (p n and Sigma+ Sigma- are computed
    # for half of the momenta) has to pair the records up one to one, or leave the pair alone when it cannot
    dup = [("p", "n", "p", "n")] * 3 + [("Sp", "Sm", "p", "Xm"), ("Sp", "Sm", "n", "X0"), ("Sp", "Sm", "n", "X0"),
                                          ("Xm", "X0", "Xm", "X0"), ("Sp", "Sm", "Sp", "Sm")]
    assert nbs.nbs_plan_selfcheck(dup) == 0
    with nbs.Nbs(L, 1, dup) as ctx:  # no image in this list: the reduced plan exists for the conjugate pairs alone
        d = to_dev(torch, S)
        ctx.load(0, d["u"], d["d"], d["s"])
        assert ctx.derived_channels() == 0 and ctx.conjugate_pairs() == 2  # p n and Xi- Xi0; Sigma+ Sigma- is not closed
    Fd = run_gpu(torch, nbs, L, S, dup)
    B = oracle.all_blocks(S, oracle.sink_names(dup))
    assert_parity(Fd, oracle.correlator_fft(L, B, dup), dup)
    dup2 = [("Sp", "Sm", "p", "Xm"), ("Sp", "Sm", "n", "X0"), ("Sp", "Sm", "L", "L"), ("Sp", "Sm", "L", "L"), ("p", "n", "p", "n"),
            ("Xm", "L", "Xm", "L"), ("S0", "p", "S0", "p")]  # four sink pairs: the pipelined kernel needs three items per task
    with nbs.Nbs(L, 1, dup2) as ctx:
        assert ctx.conjugate_pairs() == 2  # Sigma+ Sigma- (two records that are their own partners, one exchanged pair), p n
    Fd2 = run_gpu(torch, nbs, L, S, dup2)
    B = oracle.all_blocks(S, oracle.sink_names(dup2))
    assert_parity(Fd2, oracle.correlator_fft(L, B, dup2), dup2)


def test_8cubed_selected_channels(torch_cuda, nbs, oracle):
    """L = 8: the remaining power-of-two instance of the in-register FFT and of the fused inverse x-y kernel."""
    L = 8
    S = props(L, seed=19)
    chans = [("p", "n", "p", "n"), ("S0", "L", "Sp", "Sm"), ("S0", "S0", "L", "L")]
    F = run_gpu(torch_cuda, nbs, L, S, chans)
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    assert_parity(F, oracle.correlator_fft(L, B, chans), chans)


def test_smallest_lattice(torch_cuda, nbs, oracle):
    """L = 2, the smallest lattice nbs_create accepts (include/nbs.h): every momentum is its own negative, so
    the sink-swap mirror of identical baryons never applies.  All 52 channels, through the FFT path and
    through the direct shifted-sum path (row a7); L = 1 is rejected."""
    torch = torch_cuda
    L = 2
    S = props(L, seed=33)
    chans = oracle.channels52()
    with nbs.Nbs(L, 1) as ctx:
        d = to_dev(torch, S)
        ctx.load(0, d["u"], d["d"], d["s"])
        F_fft = ctx.correlator(0).cpu().numpy()
        ctx.set_direct(True)
        F_dir = ctx.correlator(0).cpu().numpy()
        torch.cuda.synchronize()
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    Fo = oracle.correlator_fft(L, B, chans)
    assert_parity(F_fft, Fo, chans)
    assert_parity(F_dir, Fo, chans)
    with pytest.raises(nbs.NbsError):
        nbs.Nbs(1, 1)


# ------------------------------------------------------------------------------ full-size dense parity (g2)
def _momentum_parity(torch, nbs, oracle, cfg, t, nq=6, seed=0):
    """All 52 channels of one dense full-size slice, in the launch configuration bench.py times, compared with the
    oracle at sampled momenta: the oracle builds its x-space blocks of every site, projects them on the sampled
    q and -q by the definition B~(q) = sum_x exp(-i q.x) B(x) and evaluates eq. 2.6's integrand
    sum_P sigma_P B~1^(P)(q) B~2^(P)(-q) there (`fourpt_momentum`); the GPU's F(r) is projected on the same q by
    the inverse of eq. 2.6, F~(q) = sum_r exp(-i q.r) F(r) (test-side DFT of the library's output).
    Returns the worst per-channel max-norm error relative to the channel's max |F~|."""
    import oracle_pool
    L, T = cfg["L"], cfg["T"]
    V = L ** 3
    S = synth.config_slice(cfg, t)
    chans = oracle.channels52()
    rng = np.random.default_rng(seed + t)
    qs = rng.choice(V, size=nq, replace=False)
    qs[0] = 1 + L * (L - 1) + L * L * 5  # one hand-picked asymmetric momentum: (1, L-1, 5)
    mq = oracle.minus_q_index(L)[qs]
    allq = np.concatenate([qs, mq])
    Bq = oracle_pool.blocks_at_momenta(L, S, oracle.sink_names(chans), allq)
    ref = np.stack([oracle.fourpt_momentum(Bq[ch[0]][:nq], Bq[ch[1]][nq:], ch).reshape(nq, 256) for ch in chans])
    with nbs.Nbs(L, T) as ctx:
        d = to_dev(torch, S)
        ctx.load(t, d["u"], d["d"], d["s"])
        F = ctx.correlator(t).reshape(len(chans) * 256, V)
        torch.cuda.synchronize()
        r = torch.arange(V, device="cuda")
        rxyz = torch.stack([r % L, (r // L) % L, r // (L * L)]).to(torch.float64)           # [3, V]
        q = torch.from_numpy(qs).cuda()
        qxyz = torch.stack([q % L, (q // L) % L, q // (L * L)], dim=1).to(torch.float64)    # [nq, 3]
        ang = (-2.0 * np.pi / L) * torch.remainder(qxyz @ rxyz, L)  # q.r mod L: exact in float64
        phase = torch.complex(torch.cos(ang), torch.sin(ang))                                # [nq, V]
        Fq = (F @ phase.T).reshape(len(chans), 256, nq).permute(0, 2, 1).cpu().numpy()       # [ch, nq, 256]
    scale = np.abs(ref).max(axis=(1, 2))
    assert scale.min() > 0
    err = np.abs(Fq - ref).max(axis=(1, 2)) / scale
    return err


def test_config1_16cubed_all_52_channels_two_slices(torch_cuda, nbs, oracle):
    """BASELINE.json configs[1] (16^3 x 32, u = d -> the isospin fast path, s): ALL 52 channels, dense Gaussian
    propagators, element by element over the whole volume against the oracle's tier B, on the first and the last
    time slice (F falls by exp(-1.4 * 31) ~ 1e-19 between them; the bar is relative per channel, reading A13)."""
    import oracle_pool
    torch = torch_cuda
    cfg = synth.CONFIGS[1]
    L, T, ts = cfg["L"], cfg["T"], [0, 31]
    chans = oracle.channels52()
    Ss = [synth.config_slice(cfg, t) for t in ts]
    assert all(S["d"] is S["u"] for S in Ss)
    Fo = oracle_pool.tierB_channels([(L, S, chans) for S in Ss])
    with nbs.Nbs(L, T) as ctx:
        for t, S, ref in zip(ts, Ss, Fo):
            d = to_dev(torch, S)
            ctx.load(t, d["u"], d["d"], d["s"])
            F = ctx.correlator(t)
            torch.cuda.synchronize()
            assert_parity(F.cpu().numpy(), ref, chans)


CFG2_SELECTED = [("p", "n", "p", "n"), ("p", "L", "S0", "p"), ("L", "L", "p", "Xm")]


@pytest.fixture(scope="module")
def cfg2_t31_reference(oracle):
    """configs[2], time slice 31: the propagators and the oracle's tier B for three channels over the whole 32^3
    volume (shared by the 32^3 and the 96^3 test below; ~90 s on 16 host cores)."""
    import oracle_pool
    cfg = synth.CONFIGS[2]
    S = synth.config_slice(cfg, 31)
    ref = oracle_pool.tierB_channels([(cfg["L"], S, CFG2_SELECTED)])[0]
    return S, ref


def test_config2_32cubed_dense_selected_channels_whole_volume(torch_cuda, nbs, oracle, cfg2_t31_reference):
    """BASELINE.json configs[2] (32^3 x 64, u != d != s, dense Gaussian propagators, all 52 channels computed as
    bench.py launches them): three channels compared element by element over all 32768 displacements with the
    oracle's tier B -- pn <- pn (two antisymmetric blocks), p Lambda <- Sigma0 p (a block without antisymmetry, a
    Sigma0 source: shared elementary correlators and the source swap) and Lambda Lambda <- p Xi- (identical sink
    baryons: half of the momenta computed, the rest mirrored).  Each covers the four accumulator layouts."""
    torch = torch_cuda
    cfg = synth.CONFIGS[2]
    L, T, t = cfg["L"], cfg["T"], 31
    S, ref = cfg2_t31_reference
    chans = oracle.channels52()
    idx = [chans.index(ch) for ch in CFG2_SELECTED]
    with nbs.Nbs(L, T) as ctx:
        d = to_dev(torch, S)
        ctx.load(t, d["u"], d["d"], d["s"])
        F = ctx.correlator(t)
        torch.cuda.synchronize()
        got = np.stack([F[i].cpu().numpy() for i in idx])
    assert_parity(got, ref, CFG2_SELECTED)


def test_config4_96cubed_tilewise_against_oracle_by_tiling(torch_cuda, nbs, oracle, cfg2_t31_reference):
    """BASELINE.json configs[4] size (96^3, 52-channel plan, tile-wise: the resident workspace would need 1.2 TB):
    the propagators are the 32^3 field of the test above repeated 3 x 3 x 3 times, for which
    F_96(r) = 27 F_32(r mod 32) (the tiling identity, pinned on the oracle in tests/test_oracle_pins.py), so the
    oracle's 32^3 tier B gives the expected value at every one of the 884736 displacements.  Channel ranges that
    hold pn <- pn, p Lambda <- Sigma0 p and Lambda Lambda <- p Xi- (an identical-baryon sink)."""
    torch = torch_cuda
    L, L0, T, t = 96, 32, 4, 1
    V = L ** 3
    S32, ref = cfg2_t31_reference
    chans = oracle.channels52()
    x = np.arange(V)
    small = (x % L) % L0 + L0 * (((x // L) % L) % L0 + L0 * ((x // (L * L)) % L0))
    d = {f: torch.from_numpy(S32[f][small]).cuda() for f in "uds"}
    small_dev = torch.from_numpy(small).cuda()
    with nbs.Nbs(L, T) as ctx:
        info = ctx.tiled_info()
        assert info["tiled"] and info["chunk_slots"] >= 2, info
        ctx.load(t, d["u"], d["d"], d["s"])
        for ch, r32 in zip(CFG2_SELECTED, ref):
            i = chans.index(ch)
            F = ctx.correlator(t, i, i + 1).reshape(256, V)
            torch.cuda.synchronize()
            want = torch.from_numpy(r32.reshape(256, L0 ** 3)).cuda()
            scale = float(want.abs().max()) * 27.0
            err = 0.0
            for a in range(0, 256, 64):  # in slabs: the gathered reference of a whole channel would be 3.6 GB more
                err = max(err, float((F[a:a + 64] - 27.0 * want[a:a + 64][:, small_dev]).abs().max()))
            assert err <= RTOL * scale, (ch, err / scale)
            del F


def test_config4_96cubed_dense_sampled_momenta(torch_cuda, nbs, oracle):
    """configs[4] itself (96^3, u = d and s, seed 5, dense): the three channels of the sink pair p Lambda on one time
    slice against the oracle at sampled momenta (see _momentum_parity: the oracle's blocks of all 884736 sites
    projected on q and -q, eq. 2.6's integrand there; the library's F(r) projected on the same q)."""
    import oracle_pool
    torch = torch_cuda
    cfg = synth.CONFIGS[4]
    L, T, t, nq = cfg["L"], cfg["T"], 2, 4
    V = L ** 3
    S = synth.config_slice(cfg, t)
    chans = oracle.channels52()
    lo, hi = 1, 4
    sel = chans[lo:hi]
    assert all(ch[:2] == ("p", "L") for ch in sel)
    rng = np.random.default_rng(96)
    qs = rng.choice(V, size=nq, replace=False)
    qs[0] = 1 + L * (L - 1) + L * L * 37
    mq = oracle.minus_q_index(L)[qs]
    Bq = oracle_pool.blocks_at_momenta(L, S, ["p", "L"], np.concatenate([qs, mq]), chunk=4096)
    ref = np.stack([oracle.fourpt_momentum(Bq[ch[0]][:nq], Bq[ch[1]][nq:], ch).reshape(nq, 256) for ch in sel])
    dd = to_dev(torch, S)
    with nbs.Nbs(L, T) as ctx:
        assert ctx.tiled_info()["tiled"]
        ctx.load(t, dd["u"], dd["d"], dd["s"])
        F = ctx.correlator(t, lo, hi).reshape((hi - lo) * 256, V)
        torch.cuda.synchronize()
        r = torch.arange(V, device="cuda")
        rxyz = torch.stack([r % L, (r // L) % L, r // (L * L)]).to(torch.float64)
        q = torch.from_numpy(qs).cuda()
        qxyz = torch.stack([q % L, (q // L) % L, q // (L * L)], dim=1).to(torch.float64)
        ang = (-2.0 * np.pi / L) * torch.remainder(qxyz @ rxyz, L)  # q.r mod L: exact in float64
        phase = torch.complex(torch.cos(ang), torch.sin(ang))
        Fq = (F @ phase.T).reshape(hi - lo, 256, nq).permute(0, 2, 1).cpu().numpy()
    scale = np.abs(ref).max(axis=(1, 2))
    err = np.abs(Fq - ref).max(axis=(1, 2)) / scale
    assert err.max() <= RTOL, (int(err.argmax()), float(err.max()))


@pytest.mark.parametrize("t", [0, 31, 63])
def test_config2_32cubed_dense_all_52_channels_sampled_momenta(torch_cuda, nbs, oracle, t):
    """configs[2], dense, all 52 channels, time slices 0, 31 and 63 (see _momentum_parity)."""
    err = _momentum_parity(torch_cuda, nbs, oracle, synth.CONFIGS[2], t)
    assert err.max() <= RTOL, (int(err.argmax()), float(err.max()))


def test_config3_32cubed_su3_dense_against_oracle(torch_cuda, nbs, oracle):
    """configs[3] (32^3, u = d = s, one array aliased three times: isospin fast path) against the oracle at sampled
    momenta, all 52 channels."""
    err = _momentum_parity(torch_cuda, nbs, oracle, synth.CONFIGS[3], 5, seed=7)
    assert err.max() <= RTOL, (int(err.argmax()), float(err.max()))


def test_blocks_dense_32cubed_sampled_sites(torch_cuda, nbs, oracle):
    """eq. 4.1 at full size with dense input: the x-space blocks of configs[2] on 48 random sites (large site
    indices included) against the oracle's blocks of those sites, one baryon of each block kind."""
    torch = torch_cuda
    cfg = synth.CONFIGS[2]
    L, T, t = cfg["L"], cfg["T"], 9
    V = L ** 3
    S = synth.config_slice(cfg, t)
    rng = np.random.default_rng(3)
    sites = np.unique(np.concatenate([rng.choice(V, size=46, replace=False), [0, V - 1]]))
    Ssub = {f: np.ascontiguousarray(S[f][sites]) for f in "uds"}
    with nbs.Nbs(L, T) as ctx:
        d = to_dev(torch, S)
        ctx.load(t, d["u"], d["d"], d["s"])
        for name in ("p", "n", "L", "S0"):
            got = ctx.blocks_x(t, name)[torch.from_numpy(sites).cuda()].cpu().numpy()
            ref = oracle.block(Ssub, name)
            assert np.abs(got - ref).max() <= RTOL * np.abs(ref).max(), name


# ------------------------------------------------------------------------------ hardening
def test_workspace_budget_slots_and_guard(torch_cuda, nbs):
    """workspace_budget_bytes: two slots when two workspaces fit, one when only one does, NBS_ENOMEM when none
    does; with ONE slot, slices loaded alternately on two streams must still give the serial results (the
    library orders the calls that share a slot, include/nbs.h nbs_num_slots)."""
    torch = torch_cuda
    L = 4
    chans = [("p", "n", "p", "n"), ("L", "L", "L", "L"), ("Xm", "L", "S0", "Xm")]
    with nbs.Nbs(L, 4, chans) as a, nbs.Nbs(L, 1, chans) as b:
        assert a.num_slots() == 2 and b.num_slots() == 1
        ws2, ws1 = a.workspace_bytes(), b.workspace_bytes()
    per_slice = ws2 - ws1
    tables = ws1 - per_slice
    assert per_slice > 0 and tables > 0
    with pytest.raises(nbs.NbsError) as e:
        nbs.Nbs(L, 4, chans, workspace_budget_bytes=tables + per_slice // 2)
    assert e.value.code == nbs.NBS_ENOMEM
    Ss = [props(L, seed=40, t=t) for t in range(4)]
    serial = [run_gpu(torch, nbs, L, Ss[t], chans, t=t, T=4) for t in range(4)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    with nbs.Nbs(L, 4, chans, workspace_budget_bytes=tables + per_slice * 3 // 2) as ctx:
        assert ctx.num_slots() == 1
        devs = [to_dev(torch, S) for S in Ss]
        torch.cuda.synchronize()
        outs = []
        for rep in range(3):  # repeat: a race would not show on every run
            outs = []
            for t in range(4):
                st = streams[t % 2]
                ctx.load(t, devs[t]["u"], devs[t]["d"], devs[t]["s"], stream=st)
                outs.append(ctx.correlator(t, stream=st))
            torch.cuda.synchronize()
            for t in range(4):
                assert np.array_equal(outs[t].cpu().numpy(), serial[t]), (rep, t)


def test_host_output_range_checked_before_launch(torch_cuda, nbs):
    """A host output larger than the device staging is refused (NBS_ENOMEM) before any kernel is enqueued."""
    L = 2
    chans = [("p", "n", "p", "n")] * 1 + [("p", "p", "p", "p"), ("n", "n", "n", "n"), ("p", "n", "p", "n")] * 40
    S = props(L, seed=41)
    with nbs.Nbs(L, 1, chans) as ctx:
        ctx.load(0, S["u"], S["d"], S["s"])
        n0 = ctx.kernel_launches()
        host = np.empty((len(chans), 4, 4, 4, 4, L ** 3), dtype=np.complex128)
        with pytest.raises(nbs.NbsError) as e:
            ctx.correlator(0, out=host)
        assert e.value.code == nbs.NBS_ENOMEM
        assert ctx.kernel_launches() == n0


def test_fp64_probe(torch_cuda, nbs):
    """nbs_probe_fp64: the register-resident mixes run and report plausible FP64 rates on a B200."""
    with nbs.Nbs(2, 1, [("p", "n", "p", "n")]) as ctx:
        dmma = ctx.probe_fp64(0, 20000)["tflops"]
        assert 10.0 < dmma < 60.0, dmma
        for mode in (1, 2, 3, 4, 5, 6, 7, 8):
            assert ctx.probe_fp64(mode, 5000)["tflops"] > 1.0
        with pytest.raises(nbs.NbsError):
            ctx.probe_fp64(9, 10)


def test_kstep_probe(torch_cuda, nbs):
    """nbs_probe_kstep: the unit code of the pipelined kernel in isolation runs for both accumulator classes and its
    time per k-step lies between the FP64-pipe bound (238 / 341 cycles per sub-partition) and a loose ceiling."""
    with nbs.Nbs(2, 1, [("p", "n", "p", "n")]) as ctx:
        for cls, floor in ((0, 238.0), (2, 341.0)):
            r = ctx.probe_kstep(cls, 8, nsteps=18, reps=50)
            assert 0.9 * floor < r["per_subpartition"] < 6 * floor, (cls, r)
            assert r["cycles_max"] >= r["cycles"]
        with pytest.raises(nbs.NbsError):
            ctx.probe_kstep(1, 8)
        with pytest.raises(nbs.NbsError):
            ctx.probe_kstep(0, 13)


# ------------------------------------------------------------------------------ tile-wise plan (configs[4], g1)
@pytest.mark.parametrize("L", [4, 6])
def test_tilewise_plan_equals_resident_plan_and_oracle(torch_cuda, nbs, oracle, L):
    """The plan of BASELINE.json configs[4] ("blocks must be contracted tile-wise, never materialised") forced on a
    small lattice by a tiny workspace budget: two-plane chunks built on demand (2 or 3 chunk buffers: evictions and
    rebuilds), one product launch per (sink pair, plane pair, plane pair), all 52 channels -- against the oracle and
    against the resident plan.  L = 6 also takes the radix-3 FFT (96 = 3 * 32).  Device and host output, and a
    channel range that cuts through sink pairs."""
    torch = torch_cuda
    V = L ** 3
    S = props(L, seed=61)
    chans = oracle.channels52()
    with nbs.Nbs(L, 1) as ctx:
        assert not ctx.tiled_info()["tiled"]
        ws_res = ctx.workspace_bytes()
        d = to_dev(torch, S)
        ctx.load(0, d["u"], d["d"], d["s"])
        F_res = ctx.correlator(0).cpu().numpy()
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    Fo = oracle.correlator_fft(L, B, chans)
    assert_parity(F_res, Fo, chans)
    # resident: B [V][34752] (compact rows; no expanded copy with the pipelined kernel) + Ft [V][52][256]; tile-wise: n chunks [V][3480] + Ft [V][6][256]
    base = ws_res - V * (34752 + 52 * 256) * 16
    for nchunks in (2, 3):
        budget = base + V * (nchunks * 3480 + 6 * 256) * 16 + V * 3480 * 8  # half a chunk of slack
        with nbs.Nbs(L, 1, workspace_budget_bytes=budget) as ctx:
            info = ctx.tiled_info()
            assert info["tiled"] and info["chunk_slots"] == nchunks, info
            d = to_dev(torch, S)
            ctx.load(0, d["u"], d["d"], d["s"])
            F = ctx.correlator(0).cpu().numpy()
            assert_parity(F, Fo, chans)
            assert_parity(F, F_res, chans)
            builds = ctx.tiled_info()["chunk_builds"]
            assert builds >= 16  # 8 baryons x 2 plane pairs at least once
            part = ctx.correlator(0, 9, 13).cpu().numpy()  # cuts the pairs (Sigma0 p) and (Lambda Lambda)
            assert np.array_equal(part, F[9:13])
            host = np.empty((3, 4, 4, 4, 4, V), dtype=np.complex128)
            ctx.correlator(0, 40, 43, out=host)
            torch.cuda.synchronize()
            assert np.array_equal(host, F[40:43])
            with pytest.raises(nbs.NbsError):
                ctx.set_direct(True)
    with pytest.raises(nbs.NbsError) as e:
        nbs.Nbs(L, 1, workspace_budget_bytes=base + V * (1 * 3480 + 6 * 256) * 16)
    assert e.value.code == nbs.NBS_ENOMEM


def test_tilewise_plan_user_channels_identical_sinks(torch_cuda, nbs, oracle):
    """Tile-wise plan on a user channel list made of identical-baryon sinks (the (0,1) tile on every momentum and its
    mirror, reading A11) and an elementary-operator channel, odd L (one self-conjugate momentum)."""
    torch = torch_cuda
    L = 3
    V = L ** 3
    S = props(L, seed=62)
    chans = [("L", "L", "L", "L"), ("L", "L", "S0", "S0"), ("S0", "S0", "Sp", "Sm"), ("p", "p", "p", "p"), ("p", "L", "p", "Xu")]
    with nbs.Nbs(L, 1, chans) as ctx:
        ws_res = ctx.workspace_bytes()
    # a budget well below the resident workspace but above two chunks + Ft + tables
    with nbs.Nbs(L, 1, chans, workspace_budget_bytes=ws_res - V * 6960 * 16) as ctx:
        assert ctx.tiled_info()["tiled"]
        d = to_dev(torch, S)
        ctx.load(0, d["u"], d["d"], d["s"])
        F = ctx.correlator(0).cpu().numpy()
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    assert_parity(F, oracle.correlator_fft(L, B, chans), chans)


def test_repeated_runs_are_bitwise_identical(torch_cuda, nbs):
    """The product kernel hands units to warps dynamically and combines their results in a fixed order, two workspace
    slots alternate and the tile-wise plan rebuilds chunks: every run of the same slice must give the same bits (a data
    race between the compute warps, the bulk-copy engine and the epilogue warps would show up here; compute-sanitizer's
    racecheck is not available on the target pool)."""
    torch = torch_cuda
    L = 8
    S = props(L, seed=71)
    d = to_dev(torch, S)
    with nbs.Nbs(L, 2) as ctx:
        ref = None
        for rep in range(6):
            t = rep % 2  # both workspace slots
            ctx.load(t, d["u"], d["d"], d["s"])
            F = ctx.correlator(t)
            torch.cuda.synchronize()
            if ref is None:
                ref = F.clone()
            else:
                assert torch.equal(F, ref), rep
    with nbs.Nbs(L, 1) as ctx:
        ws1 = ctx.workspace_bytes()
    V = L ** 3
    base = ws1 - V * (34752 + 52 * 256) * 16
    with nbs.Nbs(L, 1, workspace_budget_bytes=base + V * (2 * 3480 + 6 * 256) * 16 + V * 3480 * 8) as ctx:
        assert ctx.tiled_info()["tiled"]
        first = None
        for rep in range(2):  # chunks rebuilt and evicted on the way: same bits again
            ctx.load(0, d["u"], d["d"], d["s"])
            F = ctx.correlator(0)
            torch.cuda.synchronize()
            if first is None:
                first = F.clone()
            else:
                assert torch.equal(F, first), ("tile-wise", rep)
        # against the resident plan: the same product arithmetic, another order of the inverse FFT passes
        assert float((first - ref).abs().max()) <= 1e-13 * float(ref.abs().max())


# ------------------------------------------------------------------------------ the two product kernels
@pytest.mark.parametrize("L,same", [(4, ()), (6, ()), (4, (("d", "u"),))])
def test_pipelined_kernel_equals_one_buffer_kernel_and_oracle(torch_cuda, nbs, oracle, L, same):
    """nbs_set_pipelined: k_product_c (compact antisymmetric blocks staged as stored, load program, no barrier between
    sink pairs) and k_product_t (expanded blocks, two buffers) evaluate the same gather terms -- all 52 channels
    agree to rounding, and both match the oracle (eq. 2.6 path).  With d == u the pipelined kernel reads the blocks of
    n, Sigma-, Xi- from their partners' compact blocks with a sign."""
    torch = torch_cuda
    S = props(L, seed=77, t=1, same=same)
    chans = oracle.channels52()
    with nbs.Nbs(L, 2) as ctx:
        assert ctx.pipelined()
        ws0 = ctx.workspace_bytes()
        d = to_dev(torch, S)
        ctx.load(1, d["u"], d["d"], d["s"])
        Fp = ctx.correlator(1).clone()
        n0 = ctx.kernel_launches()
        ctx.set_pipelined(False)                      # allocates the expanded-block buffer
        assert not ctx.pipelined() and ctx.workspace_bytes() > ws0
        Fo1 = ctx.correlator(1).clone()
        n1 = ctx.kernel_launches()
        ctx.set_pipelined(True)
        Fp2 = ctx.correlator(1)
        torch.cuda.synchronize()
        assert n1 - n0 == (ctx.kernel_launches() - n1) + 1  # the one-buffer path has one more launch: the expansion pass
        assert torch.equal(Fp, Fp2)                   # bitwise reproducible, also after switching back
        scale = float(Fo1.abs().max())
        assert float((Fp - Fo1).abs().max()) <= 1e-13 * scale
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    Fo = oracle.correlator_fft(L, B, chans)
    assert_parity(Fp.cpu().numpy(), Fo, chans)
    assert_parity(Fo1.cpu().numpy(), Fo, chans)


def test_pipelined_kernel_needs_three_items(torch_cuda, nbs, oracle):
    """A plan with a single sink pair has fewer than three items per momentum pair: the library runs the one-buffer
    kernel, says so, and refuses the switch."""
    torch = torch_cuda
    chans = [("p", "n", "p", "n")]
    with nbs.Nbs(4, 1, chans) as ctx:
        assert not ctx.pipelined()
        with pytest.raises(nbs.NbsError):
            ctx.set_pipelined(True)
        S = props(4, seed=5)
        d = to_dev(torch, S)
        ctx.load(0, d["u"], d["d"], d["s"])
        F = ctx.correlator(0).cpu().numpy()
    B = oracle.all_blocks(S, oracle.sink_names(chans))
    assert_parity(F, oracle.correlator_fft(4, B, chans), chans)


def test_pipelined_kernel_user_channel_lists(torch_cuda, nbs, oracle):
    """Load programs for other channel lists: a full-full-only list (every transition waits for the previous item), a
    mixed list with elementary operators, a list whose half chain is empty (identical sink baryons only)."""
    torch = torch_cuda
    lists = [
        [("L", "L", "L", "L"), ("S0", "L", "S0", "L"), ("S0", "S0", "L", "L"), ("S0", "S0", "Sp", "Sm")],
        [("p", "L", "p", "L"), ("Sp", "n", "p", "L"), ("S0", "p", "Sp", "n"), ("Xm", "L", "Xm", "L"), ("p", "n", "p", "n")],
        [("L", "L", "L", "L"), ("S0", "S0", "S0", "S0"), ("p", "p", "p", "p")],
    ]
    for L, chans in zip((4, 3, 4), lists):
        S = props(L, seed=31 + L)
        with nbs.Nbs(L, 1, chans) as ctx:
            assert ctx.pipelined()
            d = to_dev(torch, S)
            ctx.load(0, d["u"], d["d"], d["s"])
            F = ctx.correlator(0).cpu().numpy()
        B = oracle.all_blocks(S, oracle.sink_names(chans))
        assert_parity(F, oracle.correlator_fft(L, B, chans), chans)
