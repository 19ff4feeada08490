"""The chained decoder-layer stack of BASELINE.json configs[3] as a list of program stages (plumbing only).

Per layer (reading R12; attention, activation function, norm and residual are skipped):
    q,k,v = lin(quant(h));  h2 = lin_o(quant(q));  g,u = lin(quant(h2));  h' = lin_down(quant(u))
i.e. four stages per layer, all intermediates bf16: [q|k|v] <- h, [o] <- q, [gate|up] <- h2, [down] <- u.
Nothing here computes: the stages are executed by vla_program_run (M <= 16, one persistent launch) or, for
larger M, one vla_ternary_linear call per linear (`run_stack_calls`).
"""
import torch

from . import binding as vla
from . import synth

STAGES = [("h", ["q", "k", "v"]), ("q", ["o"]), ("o", ["gate", "up"]), ("up", ["down"])]
_DIMS = {name: (K, N) for (name, K, N) in synth.STACK_LINEARS}


class Stack:
    """Device-resident weights and activation buffers of `layers` decoder layers at M tokens."""

    def __init__(self, layers, M, device="cuda", weights=None):
        self.layers, self.M, self.device = layers, M, device
        self.packed, self.beta = [], []
        for layer in range(layers):
            lw = weights[layer] if weights is not None else synth.stack_layer(layer)
            p, b = {}, {}
            for d in lw:
                w = torch.from_numpy(d["w"]).to(device)
                p[d["name"]] = vla.pack_weights(w)
                b[d["name"]] = torch.tensor([float(d["beta"])], dtype=torch.float32, device=device)
                del w
            self.packed.append(p)
            self.beta.append(b)
        # per-layer outputs (kept, so that every intermediate can be compared with the oracle)
        self.h0 = torch.zeros((M, 2560), dtype=torch.bfloat16, device=device)
        self.out = [{name: torch.zeros((M, _DIMS[name][1]), dtype=torch.bfloat16, device=device)
                     for name in _DIMS} for _ in range(layers)]
        self.packed_bytes = sum(t.numel() for p in self.packed for t in p.values())

    def set_input(self, x_bits_u16):
        import numpy as np
        t = torch.from_numpy(np.ascontiguousarray(x_bits_u16).view(np.int16)).to(self.device).view(torch.bfloat16)
        self.h0.copy_(t)

    def _input_of(self, layer, src):
        if src == "h":
            return self.h0 if layer == 0 else self.out[layer - 1]["down"]
        return self.out[layer][src]

    def stages(self):
        """Stage descriptors for vla_program_build (M <= 16)."""
        st = []
        for layer in range(self.layers):
            for (src, names) in STAGES:
                st.append(dict(
                    x=self._input_of(layer, src), M=self.M, K=_DIMS[names[0]][0],
                    depends=0 if (layer == 0 and src == "h") else 1,
                    linears=[dict(packed=self.packed[layer][n], w_scale=self.beta[layer][n], out=self.out[layer][n],
                                  N=_DIMS[n][1], out_dtype=vla.VLA_BF16) for n in names]))
        return st

    def stages_row_blocks(self, blocks):
        """The same chain as `blocks` independent chains over row blocks of the batch (a linear layer acts on every token
        row by itself), their stages interleaved: stage (layer, kind, block b) reads and writes rows [r_b, r_b+1) of the
        same tensors and waits only for the stages up to the previous kind OF ITS OWN BLOCK (depends = blocks), so that the
        grid-wide hand-offs of one block overlap the GEMMs of the others (large programs only: M / blocks > 16)."""
        M = self.M
        bounds = [(M * b // blocks) // 16 * 16 if b < blocks else M for b in range(blocks + 1)]
        st, first = [], True
        for layer in range(self.layers):
            for (src, names) in STAGES:
                for b in range(blocks):
                    r0, r1 = bounds[b], bounds[b + 1]
                    st.append(dict(
                        x=self._input_of(layer, src)[r0:r1], M=r1 - r0, K=_DIMS[names[0]][0],
                        depends=0 if first else blocks,
                        linears=[dict(packed=self.packed[layer][n], w_scale=self.beta[layer][n], out=self.out[layer][n][r0:r1],
                                      N=_DIMS[n][1], out_dtype=vla.VLA_BF16) for n in names]))
                first = False
        return st

    def compile(self, blocks=1):
        self.program = vla.compile_program(self.stages() if blocks == 1 else self.stages_row_blocks(blocks), self.device)
        return self.program

    def run_program(self):
        vla.vla_program_run(self.program)

    def alloc_call_workspace(self):
        M = self.M
        self.xq = {K: torch.empty((M, K), dtype=torch.int8, device=self.device) for K in (2560, 6912)}
        self.xs = torch.empty((M,), dtype=torch.float32, device=self.device)
        self._groups = {}

    def run_stack_calls(self):
        """One activation quant per stage and one grouped GEMM call per stage (any M; one tcgen05 launch per stage for
        M > 32, one launch per linear otherwise)."""
        M = self.M
        for layer in range(self.layers):
            for (src, names) in STAGES:
                x = self._input_of(layer, src)
                K = _DIMS[names[0]][0]
                vla.vla_act_quant(x, M, K, self.xq[K], self.xs)
                key = (layer, src)
                if key not in self._groups:
                    self._groups[key] = vla.make_linears(
                        [dict(packed=self.packed[layer][n], w_scale=self.beta[layer][n], out=self.out[layer][n],
                              N=_DIMS[n][1], out_dtype=vla.VLA_BF16) for n in names])
                vla.vla_ternary_gemm_grouped(self._groups[key], self.xq[K], self.xs, M, K)
