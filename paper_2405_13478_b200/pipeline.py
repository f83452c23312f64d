"""Host-to-host streaming wrapper over blink_grid_image: visibilities in pinned host memory in,
images in pinned host memory out, with the transfers of one chunk of time steps overlapped with the
imaging of the next on separate CUDA streams (the interleaving of "kernel executions on portions of
data ... with memory transfers" and pinned host memory the paper lists as its next optimisation,
PAPER.md:536-538).  Pure plumbing: every step of the path still runs in the CUDA kernels behind the
C ABI."""
from __future__ import annotations


class HostPipeline:
    def __init__(self, plan, n_t_max: int, chunk_t: int | None = None, depth: int = 3):
        import torch
        self.plan, self.depth = plan, depth
        # ~8 chunks per batch: small enough to overlap, large enough to fill the GPU per launch
        self.chunk_t = max(1, chunk_t if chunk_t else -(-n_t_max // 8))
        n, c = plan.n_pix, plan.n_ch
        self.vis_d = [torch.empty((self.chunk_t, c, plan.n_bl), dtype=torch.complex64, device="cuda")
                      for _ in range(depth)]
        self.img_d = [torch.empty((self.chunk_t, c, n, n), dtype=torch.float32, device="cuda")
                      for _ in range(depth)]
        self.s_in, self.s_cmp, self.s_out = (torch.cuda.Stream() for _ in range(3))
        plan.reserve(self.chunk_t)

    def run(self, vis_h, img_h):
        """vis_h: pinned complex64 [n_t, n_ch, n_bl]; img_h: pinned float32 [n_t, n_ch, N, N].
        Asynchronous w.r.t. the host; ordered after/before the current stream."""
        import torch
        cur = torch.cuda.current_stream()
        start = torch.cuda.Event()
        start.record(cur)
        for s in (self.s_in, self.s_cmp, self.s_out):
            s.wait_event(start)
        n_t = vis_h.shape[0]
        in_done = [None] * self.depth
        cmp_done = [None] * self.depth
        out_done = [None] * self.depth
        for i, t0 in enumerate(range(0, n_t, self.chunk_t)):
            t1, b = min(n_t, t0 + self.chunk_t), i % self.depth
            k = t1 - t0
            with torch.cuda.stream(self.s_in):
                if cmp_done[b] is not None:
                    self.s_in.wait_event(cmp_done[b])          # vis_d[b] has been consumed
                self.vis_d[b][:k].copy_(vis_h[t0:t1], non_blocking=True)
                in_done[b] = torch.cuda.Event()
                in_done[b].record(self.s_in)
            with torch.cuda.stream(self.s_cmp):
                self.s_cmp.wait_event(in_done[b])
                if out_done[b] is not None:
                    self.s_cmp.wait_event(out_done[b])         # img_d[b] has been copied out
                self.plan.grid_image(self.vis_d[b][:k], self.img_d[b][:k], stream=self.s_cmp)
                cmp_done[b] = torch.cuda.Event()
                cmp_done[b].record(self.s_cmp)
            with torch.cuda.stream(self.s_out):
                self.s_out.wait_event(cmp_done[b])
                img_h[t0:t1].copy_(self.img_d[b][:k], non_blocking=True)
                out_done[b] = torch.cuda.Event()
                out_done[b].record(self.s_out)
        for s in (self.s_in, self.s_cmp, self.s_out):
            done = torch.cuda.Event()
            done.record(s)
            cur.wait_event(done)
        return img_h
