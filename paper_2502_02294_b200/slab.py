"""slab.py -- the exchange layer of the slab decomposition.

The paper: hydro "can be parallelized by splitting the volume ... communication limited to the boundaries", while the
particle-mesh gravity needs FFTs "over the entire volume".  north_star fixes one GPU and no sharding, and
this pool gives one GPU per call, so what is built here is the part that can be proven without a second GPU: WHAT moves
between ranks, in which layout, and that it reassembles to the single-rank result.  One process per GPU, torch.distributed
(NCCL over NVLink on B200s, gloo on the CPU in tests/test_slab_exchange.py); tensors stay on whatever device they are on.

Partition: rank r of P owns the mesh planes z in [r nz, (r + 1) nz), nz = N / P, of every field ([z][y][x] as in the
library), and the particles whose z lies in that range.  Per coupled step (S1-S4):

  S1  deposit            particles within half a cell of a slab face touch one plane of the neighbour: deposit into a
                         slab padded by 1 plane on each side, then `halo_reduce` (1 plane each way, added)
  S2  Poisson solve      per-plane 2-D transforms are local (the library's x and y passes); one `transpose_z_to_x`
                         (all-to-all) makes z local for the fused z pass (transform, Green multiply, inverse); three
                         `transpose_x_to_z` bring g'_x, g'_y, g'_z back: 4 all-to-alls of 4 B/cell each
  S3  gather, kick-drift `halo_exchange` of g' (1 plane each way), then `migrate` (particles that left the slab)
  S4  sweeps             x and y sweeps are slab-local; the z sweep needs `halo_exchange` of the five fields and g'_z by
                         3 planes (forward) / 4 planes (adjoint) each way
  reverse pass           the transposes of the above: `halo_reduce` where the forward has `halo_exchange` and vice versa,
                         the same all-to-alls with the roles of the two layouts swapped

The compute between the exchanges is the library's existing kernels on a slab-shaped mesh (nz + 2 halo planes instead of
N): that launch geometry is NOT built (every kernel assumes a cubic periodic box), which is why this module carries a
plain torch stand-in for the per-rank transforms in `poisson_slab` -- used by the test only, to prove the exchange.
`comm_bytes_per_step` is the model DESIGN.md quotes against NVLink bandwidth.
"""
from __future__ import annotations

import math

import torch
import torch.distributed as dist


class Slab:
    """Layout and exchange operations of one rank.  group=None: the default process group."""

    def __init__(self, N: int, group=None):
        self.group = group
        self.P = dist.get_world_size(group)
        self.rank = dist.get_rank(group)
        if N % self.P:
            raise ValueError(f"grid side {N} is not a multiple of the world size {self.P}")
        self.N, self.nz = N, N // self.P
        self.z0 = self.rank * self.nz
        self.up = (self.rank + 1) % self.P          # owner of the planes above mine (periodic)
        self.down = (self.rank - 1) % self.P
        self.bytes_sent = 0                          # payload this rank handed to the transport (the test checks the model)

    # ------------------------------------------------------------------------------------------------ halos ----
    def _swap(self, to_up: torch.Tensor, to_down: torch.Tensor):
        """Send `to_up` to the rank above and `to_down` to the rank below; return (from_below, from_above)."""
        to_up, to_down = to_up.contiguous(), to_down.contiguous()
        from_below, from_above = torch.empty_like(to_up), torch.empty_like(to_down)
        self.bytes_sent += (to_up.numel() + to_down.numel()) * to_up.element_size()
        if self.P == 1:
            from_below.copy_(to_up); from_above.copy_(to_down)
            return from_below, from_above
        ops = [dist.P2POp(dist.isend, to_up, self.up, self.group), dist.P2POp(dist.irecv, from_below, self.down, self.group),
               dist.P2POp(dist.isend, to_down, self.down, self.group), dist.P2POp(dist.irecv, from_above, self.up, self.group)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        return from_below, from_above

    def halo_exchange(self, f: torch.Tensor, h: int) -> torch.Tensor:
        """f (..., nz, N, N) -> (..., nz + 2h, N, N): h planes of each neighbour around my slab (periodic in z)."""
        assert f.shape[-3] == self.nz and 0 < h <= self.nz
        from_below, from_above = self._swap(f[..., self.nz - h:, :, :], f[..., :h, :, :])
        return torch.cat([from_below, f, from_above], dim=-3)

    def halo_reduce(self, fp: torch.Tensor, h: int) -> torch.Tensor:
        """Transpose of halo_exchange: fp (..., nz + 2h, N, N) -> (..., nz, N, N), the pad planes ADDED onto the
        neighbours' outermost interior planes (deposit into a padded slab; cotangents of exchanged halos)."""
        assert fp.shape[-3] == self.nz + 2 * h
        from_below, from_above = self._swap(fp[..., self.nz + h:, :, :], fp[..., :h, :, :])
        out = fp[..., h:self.nz + h, :, :].clone()
        out[..., :h, :, :] += from_below            # what the rank below deposited above its top face
        out[..., self.nz - h:, :, :] += from_above
        return out

    # -------------------------------------------------------------------------------------------- particles ----
    def owner_of(self, z: torch.Tensor) -> torch.Tensor:
        """Rank that owns position z (grid units, [0, N)): floor(z / nz); the very test `migrate` applies."""
        return torch.clamp(torch.floor(z / self.nz).to(torch.int64), 0, self.P - 1)

    def migrate(self, part: torch.Tensor, return_route: bool = False):
        """part (k, n), k >= 3: rows 0-2 are positions (grid units), the rest travels with them (velocities, ids, ...).
        Returns the particles this rank owns after the exchange, grouped by source rank in rank order.
        Counts first, then the payload as one all-to-all with ragged splits.  return_route: also the routing record that
        `migrate_back` needs (the transpose: cotangents return to the rank and the slot their particle came from)."""
        k, n = part.shape
        owner = self.owner_of(part[2])
        order = torch.argsort(owner, stable=True)
        send = part[:, order].t().contiguous()                       # (n, k) grouped by destination
        counts = torch.bincount(owner, minlength=self.P)
        recv_counts = counts.clone()
        if self.P > 1:
            dist.all_to_all_single(recv_counts, counts, group=self.group)
            out = torch.empty((int(recv_counts.sum()), k), dtype=part.dtype, device=part.device)
            self.bytes_sent += int(counts.sum() - counts[self.rank]) * k * part.element_size()
            dist.all_to_all_single(out, send, output_split_sizes=recv_counts.tolist(), input_split_sizes=counts.tolist(),
                                   group=self.group)
        else:
            out = send
        res = out.t().contiguous()
        return (res, (order, counts.tolist(), recv_counts.tolist(), n)) if return_route else res

    def migrate_back(self, cot: torch.Tensor, route) -> torch.Tensor:
        """Transpose of migrate: cot (k, n_after) in the order migrate returned -> (k, n_before) in the order migrate was given."""
        order, counts, recv_counts, n = route
        k = cot.shape[0]
        send = cot.t().contiguous()
        if self.P > 1:
            back = torch.empty((n, k), dtype=cot.dtype, device=cot.device)
            self.bytes_sent += (sum(recv_counts) - recv_counts[self.rank]) * k * cot.element_size()
            dist.all_to_all_single(back, send, output_split_sizes=counts, input_split_sizes=recv_counts, group=self.group)
        else:
            back = send
        res = torch.empty_like(back)
        res[order] = back                                             # undo the grouping by destination
        return res.t().contiguous()

    # ------------------------------------------------------------------------------------------- transposes ----
    def transpose_z_to_x(self, a: torch.Tensor) -> torch.Tensor:
        """a (nz, N, M) with M a multiple of P (z local slab, all of x) -> (N, N, M / P) (all of z, my share of x).
        One all-to-all: block (q, r) of the P x P decomposition goes from rank r to rank q."""
        nz, N, M = a.shape
        assert nz == self.nz and M % self.P == 0
        m = M // self.P
        send = a.reshape(nz, N, self.P, m).permute(2, 0, 1, 3).contiguous()         # [dest][z][y][x']
        recv = torch.empty_like(send)                                                # [source][z][y][x']
        self.bytes_sent += send.numel() * send.element_size() * (self.P - 1) // self.P
        if self.P == 1:
            recv.copy_(send)
        else:
            dist.all_to_all_single(recv, send, group=self.group)
        return recv.reshape(self.P * nz, N, m)

    def transpose_x_to_z(self, b: torch.Tensor) -> torch.Tensor:
        """Inverse of transpose_z_to_x: b (N, N, m) -> (nz, N, m P)."""
        Nz, N, m = b.shape
        assert Nz == self.N
        send = b.reshape(self.P, self.nz, N, m).contiguous()                         # [dest = z block][z][y][x']
        recv = torch.empty_like(send)                                                # [source = x block][z][y][x']
        self.bytes_sent += send.numel() * send.element_size() * (self.P - 1) // self.P
        if self.P == 1:
            recv.copy_(send)
        else:
            dist.all_to_all_single(recv, send, group=self.group)
        return recv.permute(1, 2, 0, 3).reshape(self.nz, N, self.P * m)

    # ----------------------------------------------------------------- the Poisson solve across slabs (S2) ----
    def poisson_slab(self, delta: torch.Tensor, A: float, box: float) -> torch.Tensor:
        """g'_d (3, nz, N, N) from my slab of delta_tot (nz, N, N): reading R12 of DESIGN.md (Green -1/k^2, gradient i k,
        zero mode 0, the Nyquist component of k_d zeroed).  The per-rank transforms here are torch.fft stand-ins for the
        library's x / y passes and fused z pass; the four all-to-alls are the product's."""
        N, P = self.N, self.P
        nxh = N // 2 + 1
        M = P * math.ceil(nxh / P)                                   # pad the half spectrum to a multiple of P
        spec = torch.fft.rfft2(delta.to(torch.float64), dim=(-2, -1))               # (nz, N, nxh), y and x local
        pad = torch.zeros((self.nz, N, M), dtype=spec.dtype, device=spec.device)
        pad[..., :nxh] = spec
        # complex payloads travel as two real meshes (re, im)
        re = self.transpose_z_to_x(pad.real.contiguous())
        im = self.transpose_z_to_x(pad.imag.contiguous())
        colz = torch.fft.fft(torch.complex(re, im), dim=0)                          # (N, N, m): z now local
        m = M // P
        kf = 2.0 * math.pi / box
        nfreq = torch.fft.fftfreq(N, d=1.0 / N, device=delta.device, dtype=torch.float64)
        nz_ = nfreq[:, None, None]
        ny_ = nfreq[None, :, None]
        nx_ = (torch.arange(m, device=delta.device, dtype=torch.float64) + self.rank * m)[None, None, :]
        k2 = kf * kf * (nx_ * nx_ + ny_ * ny_ + nz_ * nz_)
        inv = torch.where(k2 > 0, 1.0 / torch.where(k2 > 0, k2, torch.ones_like(k2)), torch.zeros_like(k2))
        live = (nx_ < nxh).to(torch.float64)                          # padded columns carry nothing
        out = []
        for n_d in (nx_, ny_, nz_):
            nt = torch.where(n_d.abs() == N // 2, torch.zeros_like(n_d), n_d)
            gz = torch.fft.ifft(1j * kf * nt * A * inv * live * colz, dim=0)        # g^_d = i k~_d A delta^ / k^2
            back = torch.complex(self.transpose_x_to_z(gz.real.contiguous()), self.transpose_x_to_z(gz.imag.contiguous()))
            out.append(torch.fft.irfft2(back[..., :nxh], s=(N, N), dim=(-2, -1)))
        return torch.stack(out)


    def poisson_slab_vjp(self, gb: torch.Tensor, A: float, box: float) -> torch.Tensor:
        """Transpose of poisson_slab: delta_b (nz, N, N) = sum_d G_d^T g_b,d.  G_d = F^-1 (i k~_d A / k^2) F with an odd
        imaginary symbol, so G_d^T = -G_d: three all-to-alls in, one out (the roles of the layouts swapped)."""
        N, P = self.N, self.P
        nxh = N // 2 + 1
        M = P * math.ceil(nxh / P)
        m = M // P
        kf = 2.0 * math.pi / box
        nfreq = torch.fft.fftfreq(N, d=1.0 / N, device=gb.device, dtype=torch.float64)
        nz_ = nfreq[:, None, None]
        ny_ = nfreq[None, :, None]
        nx_ = (torch.arange(m, device=gb.device, dtype=torch.float64) + self.rank * m)[None, None, :]
        k2 = kf * kf * (nx_ * nx_ + ny_ * ny_ + nz_ * nz_)
        inv = torch.where(k2 > 0, 1.0 / torch.where(k2 > 0, k2, torch.ones_like(k2)), torch.zeros_like(k2))
        live = (nx_ < nxh).to(torch.float64)
        acc = None
        for d, n_d in enumerate((nx_, ny_, nz_)):
            spec = torch.fft.rfft2(gb[d].to(torch.float64), dim=(-2, -1))
            pad = torch.zeros((self.nz, N, M), dtype=spec.dtype, device=spec.device)
            pad[..., :nxh] = spec
            colz = torch.fft.fft(torch.complex(self.transpose_z_to_x(pad.real.contiguous()),
                                               self.transpose_z_to_x(pad.imag.contiguous())), dim=0)
            nt = torch.where(n_d.abs() == N // 2, torch.zeros_like(n_d), n_d)
            term = -(1j * kf * nt * A * inv * live) * colz
            acc = term if acc is None else acc + term
        dz = torch.fft.ifft(acc, dim=0)
        back = torch.complex(self.transpose_x_to_z(dz.real.contiguous()), self.transpose_x_to_z(dz.imag.contiguous()))
        return torch.fft.irfft2(back[..., :nxh], s=(N, N), dim=(-2, -1))


def comm_bytes_per_step(N: int, P: int, n_part_cross: float = 0.0, adjoint: bool = False) -> dict:
    """Payload each rank sends per coupled step (fp32), by phase; n_part_cross = particles leaving a slab per step.
    Forward: the S1-S4 exchanges listed in the module docstring.  adjoint=True: the step VJP's (the same exchanges
    transposed; 4-plane halos for the z sweep, cotangents of g' reduced instead of g' exchanged)."""
    plane = 4 * N * N
    a2a = lambda n_fields: n_fields * 4 * N * N * (N // P) * (P - 1) // P         # one all-to-all of n real meshes
    half = lambda: 2 * a2a(1) * (P * math.ceil((N // 2 + 1) / P)) / N              # a padded half spectrum, (re, im)
    hz = 4 if adjoint else 3
    d = {
        "deposit_halo_reduce": 2 * 1 * plane,
        "poisson_all_to_all": 4 * half(),
        "gprime_halo": 2 * 1 * 3 * plane,
        "migrate": n_part_cross * 24,
        "z_sweep_halo": 2 * hz * (5 + 1) * plane * (2 if adjoint else 1),          # adjoint: state + cotangent in, halos of both
    }
    d["total"] = sum(d.values())
    return d
