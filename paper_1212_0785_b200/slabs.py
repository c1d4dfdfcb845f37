"""Domain decomposition in t with a one-site halo ("multi-GPU (parallel
architecture) support", "overlapping communications and computation ... is work in progress").

The arithmetic stays in libqcdmd (slab lattices: qcd_lattice_create_slab; transport kernel: qcd_copy_timeslices);
this module is the plumbing above it, which is torch.distributed's job in this build:

  partition(Lt, n)        host logic: the n slabs (t_begin, t_count) of a lattice of Lt timeslices
  SlabComm                who the neighbours are, face messages over torch.distributed (NCCL on GPUs, gloo in the
                          CPU tests), reductions combined in FIXED RANK ORDER (deterministic)
  DistSlab                one slab per process: fields, halo exchange, leapfrog, observables
  SlabSet                 all slabs in ONE process on one GPU: the same schedule with qcd_copy_timeslices writing
                          straight into the neighbour's halo (what peer pointers over NVLink would do), used by the
                          single-GPU tests, and with the interior / boundary split on two streams

One halo exchange per force evaluation: the lower neighbour's last interior timeslice goes to te = 0 (all four links:
U_mu(x - t) and the corner links U_t(x + mu - t)), the upper neighbour's first interior timeslice to te = n + 1
(the three spatial links U_nu(x + t); mu_mask 0x7).  Momenta never travel.  The generator is keyed on the global
site, so refresh and hot start need no exchange at all.
"""
import torch

MASK_ALL, MASK_SPATIAL = 0xF, 0x7


def partition(Lt, n):
    """n slabs of even length covering 0..Lt-1 in order, as equal as possible: [(t_begin, t_count)]"""
    if Lt % 2 or n < 1 or 2 * n > Lt:
        raise ValueError("need an even Lt and at most Lt/2 slabs")
    pairs, rest = divmod(Lt // 2, n)
    out, t = [], 0
    for r in range(n):
        c = 2 * (pairs + (1 if r < rest else 0))
        out.append((t, c))
        t += c
    return out


def ordered_sum(parts):
    """sum of per-rank partial results in rank order (Python floats / tensors): the same bits on every rank and run"""
    acc = parts[0]
    for p in parts[1:]:
        acc = acc + p
    return acc


class SlabComm:
    """Neighbours and messages of rank `rank` of `world` slabs, periodic in t.  `dist` is torch.distributed (already
    initialised) or None for a single slab (the lattice's own periodic wrap)."""

    def __init__(self, rank, world, dist=None):
        self.rank, self.world, self.dist = rank, world, dist
        self.lower, self.upper = (rank - 1) % world, (rank + 1) % world

    def exchange(self, to_lower, to_upper):
        """send one face to each neighbour, receive theirs: returns (from_lower, from_upper).  The two messages may
        differ in size (the face sent down carries three links, the one sent up four).  When both neighbours are the
        same rank (world = 2) gloo keeps the messages apart by tag; NCCL ignores tags and matches the sends and
        receives of a pair of ranks in the order they were posted, which is why the order below is the same on both
        sides: up-going face first (my first send, the peer's first receive), down-going face second.
        Device tensors over a CPU-only backend (gloo: the two-processes-on-one-GPU test) are staged through host
        memory; over NCCL they travel as they are."""
        if self.world == 1:
            return to_upper.clone(), to_lower.clone()
        d = self.dist
        dev = to_lower.device
        staged = self._staged(to_lower)
        if staged:
            to_lower, to_upper = to_lower.cpu(), to_upper.cpu()
        from_lower, from_upper = torch.empty_like(to_upper), torch.empty_like(to_lower)
        ops = [d.P2POp(d.isend, to_upper, self.upper, tag=0), d.P2POp(d.isend, to_lower, self.lower, tag=1),
               d.P2POp(d.irecv, from_lower, self.lower, tag=0), d.P2POp(d.irecv, from_upper, self.upper, tag=1)]
        for r in d.batch_isend_irecv(ops):
            r.wait()
        if staged:
            from_lower, from_upper = from_lower.to(dev), from_upper.to(dev)
        return from_lower, from_upper

    def _staged(self, t):
        """device tensors over a CPU-only backend go through host memory (see exchange)"""
        return t.device.type == "cuda" and self.dist.get_backend() == "gloo"

    def combine(self, local):
        """all ranks' values of a small tensor, summed in rank order (one all_gather; no rank-dependent order)"""
        if self.world == 1:
            return local.clone()
        if self._staged(local):
            return self.combine(local.cpu()).to(local.device)
        parts = [torch.empty_like(local) for _ in range(self.world)]
        self.dist.all_gather(parts, local)
        return ordered_sum(parts)

    def gather_concat(self, local):
        """per-timeslice values of every rank, concatenated in rank order = global timeslice order"""
        if self.world == 1:
            return local.clone()
        if self._staged(local):
            return self.gather_concat(local.cpu()).to(local.device)
        sizes = [torch.zeros(1, dtype=torch.int64, device=local.device) for _ in range(self.world)]
        self.dist.all_gather(sizes, torch.tensor([local.numel()], dtype=torch.int64, device=local.device))
        m = int(max(s.item() for s in sizes))
        pad = torch.zeros(m, dtype=local.dtype, device=local.device)
        pad[: local.numel()] = local
        parts = [torch.empty_like(pad) for _ in range(self.world)]
        self.dist.all_gather(parts, pad)
        return torch.cat([p[: int(s.item())] for p, s in zip(parts, sizes)])


class _SlabOps:
    """what one slab does between exchanges (shared by DistSlab and SlabSet)"""

    def __init__(self, qcd, global_dims, t_begin, t_count, dtype):
        self.qcd, self.dtype = qcd, dtype
        self.lat = qcd.Lattice(global_dims, slab=(t_begin, t_count))
        self.t_begin, self.n = t_begin, t_count
        self.U, self.P = self.lat.new_matrix_field(dtype), self.lat.new_matrix_field(dtype)
        self.ws = self.lat.new_workspace()
        self.face_lat = qcd.Lattice(tuple(global_dims[:3]) + (2,))  # one timeslice of links as a contiguous field
        self.Vs = global_dims[0] * global_dims[1] * global_dims[2]
        # boundary / interior split: the inner timeslices need no halo
        self.inner = self.lat.view_t(2, t_count) if t_count >= 4 else None
        self.edges = [self.lat.view_t(1, 2), self.lat.view_t(t_count, t_count + 1)] if t_count >= 4 else None

    def start(self, seed, sigma):
        self.qcd.qcd_hot_start(self.lat, self.U, seed, sigma)
        self.qcd.qcd_mom_refresh(self.lat, self.P, seed)

    # A face is one timeslice of links.  qcd_copy_timeslices moves it between the slab and timeslice 0 of `face_lat`,
    # a field of two timeslices (the smallest lattice the library has), and only the part of that field that holds
    # timeslice 0 goes on the wire: in the device layout (include/qcd.h) its even sites are the checkerboard indices
    # [0, Vs/2) and its odd ones [Vs, Vs + Vs/2), i.e. two runs of 32-site chunks, and a face without time-like links
    # (mask 0x7) needs the first 27 of the 36 units per site.  Per face that is about Vs x 72 (54) reals instead of
    # the 2 Vs x 72 of the whole two-timeslice field.
    def _face_chunks(self):
        if getattr(self, "_chunks", None) is None:
            h = self.Vs // 2
            idx = sorted(set(range(0, (h + 31) // 32)) | set(range(self.Vs // 32, (self.Vs + h - 1) // 32 + 1)))
            self._chunks = torch.tensor(idx, dtype=torch.int64, device="cuda")
        return self._chunks

    @staticmethod
    def _face_units(mask):
        return 27 if mask == MASK_SPATIAL else 36

    def face(self, te, mask, stream=None):
        """the links `mask` of stored timeslice te as a message: [chunks of timeslice 0][units][32][2], contiguous"""
        buf = self.face_lat.new_matrix_field(self.dtype)
        self.qcd.qcd_copy_timeslices(self.lat, self.U, te, self.face_lat, buf, 0, 1, 72, mask, stream)
        return buf[self._face_chunks(), : self._face_units(mask)].contiguous()

    def put_face(self, msg, te, mask, stream=None):
        buf = self.face_lat.new_matrix_field(self.dtype)
        buf[self._face_chunks(), : self._face_units(mask)] = msg
        self.qcd.qcd_copy_timeslices(self.face_lat, buf, 0, self.lat, self.U, te, 1, 72, mask, stream)

    def gather(self, which):
        """the interior timeslices of this slab as a canonical host array [t_count * Vs, 4, 3, 3]"""
        a = self.qcd.field_to_host(self.lat, self.U if which == "U" else self.P)
        return a.reshape(self.n + 2, self.Vs, 4, 3, 3)[1: self.n + 1].reshape(-1, 4, 3, 3)

    def observables(self):
        """per interior timeslice: plaquette average and K = sum |P_ij|^2 (device tensors of length t_count)"""
        qcd = self.qcd
        Lt = self.n + 2
        avg = torch.zeros(1, dtype=torch.float64, device="cuda")
        per_t = torch.zeros(Lt, dtype=torch.float64, device="cuda")
        kt = torch.zeros(Lt, dtype=torch.float64, device="cuda")
        qcd.qcd_plaquette(self.lat, self.U, avg, per_t, self.ws)
        qcd.qcd_sum_multi(self.lat, qcd.SUM_NORM2, 72, self.P, None, Lt, kt, self.ws)
        return per_t[1: self.n + 1].clone(), kt[1: self.n + 1].clone()


class DistSlab(_SlabOps):
    """one slab per process; halos travel through torch.distributed"""

    def __init__(self, qcd, global_dims, comm, dtype=torch.float64):
        t_begin, t_count = partition(global_dims[3], comm.world)[comm.rank]
        super().__init__(qcd, global_dims, t_begin, t_count, dtype)
        self.comm = comm

    def exchange(self):
        lo, up = self.comm.exchange(self.face(1, MASK_SPATIAL), self.face(self.n, MASK_ALL))
        self.put_face(lo, 0, MASK_ALL)
        self.put_face(up, self.n + 1, MASK_SPATIAL)

    def leapfrog(self, beta, eps, nsteps):
        qcd = self.qcd
        qcd.qcd_force_mom_update(self.lat, self.U, self.P, beta, 0.5 * eps)
        for k in range(nsteps):
            qcd.qcd_link_update(self.lat, self.P, self.U, eps, reunit=True)
            self.exchange()
            qcd.qcd_force_mom_update(self.lat, self.U, self.P, beta, 0.5 * eps if k == nsteps - 1 else eps)

    def global_observables(self, beta):
        """(plaquette, K, per-timeslice plaquette of the whole lattice), ranks combined in fixed order"""
        per_t, kt = self.observables()
        plaq_t = self.comm.gather_concat(per_t)
        K = self.comm.combine(kt.sum().reshape(1))
        return plaq_t.mean().item(), K.item(), plaq_t


class SlabSet:
    """all slabs of a lattice in one process on one GPU: qcd_copy_timeslices writes straight into the neighbour's
    halo, as a peer pointer would over NVLink.  overlap = True: the halos travel on a second stream while the force
    of the inner timeslices runs; the two boundary timeslices follow."""

    def __init__(self, qcd, global_dims, nslabs, dtype=torch.float64):
        self.qcd, self.dims = qcd, tuple(global_dims)
        self.slabs = [_SlabOps(qcd, global_dims, tb, tc, dtype) for tb, tc in partition(global_dims[3], nslabs)]
        self.comm_stream = torch.cuda.Stream()

    def start(self, seed, sigma):
        for s in self.slabs:
            s.start(seed, sigma)

    def exchange(self, stream=None):
        n = len(self.slabs)
        for r, s in enumerate(self.slabs):
            up, lo = self.slabs[(r + 1) % n], self.slabs[(r - 1) % n]
            # my last interior timeslice -> upper neighbour's lower halo; my first -> lower neighbour's upper halo
            self.qcd.qcd_copy_timeslices(s.lat, s.U, s.n, up.lat, up.U, 0, 1, 72, MASK_ALL, stream)
            self.qcd.qcd_copy_timeslices(s.lat, s.U, 1, lo.lat, lo.U, lo.n + 1, 1, 72, MASK_SPATIAL, stream)

    def kick(self, beta, eps, overlap):
        qcd = self.qcd
        if not overlap or any(s.inner is None for s in self.slabs):
            self.exchange()
            for s in self.slabs:
                qcd.qcd_force_mom_update(s.lat, s.U, s.P, beta, eps)
            return
        main = torch.cuda.current_stream()
        self.comm_stream.wait_stream(main)
        with torch.cuda.stream(self.comm_stream):
            self.exchange(self.comm_stream)
        for s in self.slabs:  # inner timeslices: no halo needed, runs while the faces travel
            qcd.qcd_force_mom_update(s.inner, s.U, s.P, beta, eps)
        main.wait_stream(self.comm_stream)
        for s in self.slabs:
            for v in s.edges:
                qcd.qcd_force_mom_update(v, s.U, s.P, beta, eps)

    def push_update(self, eps, overlap):
        """link update of every slab fused with the halo transport (qcd_link_update_push): the thread that computes a
        link of a boundary timeslice also stores it into the neighbour's halo.  overlap = True: the boundary
        timeslices go first, so their stores travel while the inner timeslices are updated"""
        n = len(self.slabs)
        views = (lambda s: list(s.edges) + [s.inner]) if overlap and all(s.inner is not None for s in self.slabs) \
            else (lambda s: [s.lat])
        for which in range(len(views(self.slabs[0]))):
            for r, s in enumerate(self.slabs):
                up, lo = self.slabs[(r + 1) % n], self.slabs[(r - 1) % n]
                self.qcd.qcd_link_update_push(views(s)[which], s.P, s.U, eps, True, lo.lat, lo.U, up.lat, up.U)

    def force(self, beta, eps):
        for s in self.slabs:
            self.qcd.qcd_force_mom_update(s.lat, s.U, s.P, beta, eps)

    def leapfrog(self, beta, eps, nsteps, overlap=False, fused=False):
        """fused = False: link update, then qcd_copy_timeslices into the neighbours' halos, then the force;
        fused = True: the link update stores the boundary timeslices into the neighbours' halos itself"""
        self.kick(beta, 0.5 * eps, overlap)  # halos are valid after start(): the exchange inside is a no-op in effect
        for k in range(nsteps):
            e = 0.5 * eps if k == nsteps - 1 else eps
            if fused:
                self.push_update(eps, overlap)
                self.force(beta, e)
            else:
                for s in self.slabs:
                    self.qcd.qcd_link_update(s.lat, s.P, s.U, eps, reunit=True)
                self.kick(beta, e, overlap)

    def leapfrog_single_pass(self, beta, eps, nsteps, overlap=False):
        """the leapfrog of single-pass steps (qcd_leapfrog_single_pass regrouping) on every slab, the halo transport
        done by the step kernel itself (qcd_md_step_single_pass_push): each step reads a slab's field with valid halos
        and writes the second field of the slab and, for the boundary timeslices, of its neighbours.  overlap = True:
        the boundary timeslices are launched first, so their stores travel while the inner timeslices are computed"""
        qcd, n = self.qcd, len(self.slabs)
        cur = [s.U for s in self.slabs]
        oth = [s.lat.new_matrix_field(s.dtype) for s in self.slabs]
        split = overlap and all(s.inner is not None for s in self.slabs)
        for k in range(nsteps):
            for which in range(3 if split else 1):
                for r, s in enumerate(self.slabs):
                    up, lo = (r + 1) % n, (r - 1) % n
                    view = (list(s.edges) + [s.inner])[which] if split else s.lat
                    qcd.qcd_md_step_single_pass_push(view, cur[r], s.P, oth[r], beta, 0.5 * eps if k == 0 else eps, eps,
                                                     self.slabs[lo].lat, oth[lo], self.slabs[up].lat, oth[up])
            cur, oth = oth, cur
        for r, s in enumerate(self.slabs):
            qcd.qcd_force_mom_update(s.lat, cur[r], s.P, beta, 0.5 * eps)
            if cur[r] is not s.U:
                s.U.copy_(cur[r])

    def gather(self, which):
        """interior timeslices of every slab as one canonical host array [V,4,3,3] of the global lattice"""
        import numpy as np
        out = []
        for s in self.slabs:
            out.append(s.gather(which))
        return np.concatenate(out)

    def global_observables(self):
        per_t, kt = zip(*(s.observables() for s in self.slabs))
        plaq_t = torch.cat(per_t)
        K = ordered_sum([k.sum() for k in kt])
        return plaq_t.mean().item(), K.item(), plaq_t
