"""Independent float64 restatement of Domino's equations out of LIBRARY routines
(torch.nn.GRUCell, F.silu, F.linear, torch.log_softmax) -- used to pin the C oracle, never by
the product.  PAPER.md:68-78 (Sec. 2.3), PAPER.md:87 (q_Domino = softmax(L_base + dL))."""
import torch
import torch.nn.functional as F


class TorchRef:
    def __init__(self, w: dict):
        self.E = w["embed"].double()
        self.W1 = w["corr_w1"].double()
        self.W2 = w["corr_w2"].double()
        g = w["gru_w_hh"].shape[1]
        d = w["embed"].shape[1]
        self.g, self.d = g, d
        self.cell = torch.nn.GRUCell(d, g, bias=False, dtype=torch.float64)
        with torch.no_grad():
            self.cell.weight_ih.copy_(w["gru_w_ih"].double())
            self.cell.weight_hh.copy_(w["gru_w_hh"].double())

    @torch.no_grad()
    def advance(self, S, token):
        return self.cell(self.E[int(token)][None], S[None])[0]

    @torch.no_grad()
    def s0(self, root):
        return self.advance(torch.zeros(self.g, dtype=torch.float64), root)

    @torch.no_grad()
    def corrected_logits(self, L_base_i, H_i, S):
        """Full-vocabulary L_i = L_i^base + W2 SiLU(W1 [H_i; S])."""
        a = F.silu(F.linear(torch.cat([H_i.double(), S]), self.W1))
        return L_base_i.double() + F.linear(a, self.W2)

    @torch.no_grad()
    def slice_logprobs(self, L_base_i, H_i, S, cand, T_eff=1.0):
        z = self.corrected_logits(L_base_i, H_i, S)[cand.long()] / T_eff
        return torch.log_softmax(z, dim=0)


def order_desc(values: torch.Tensor, tokens: torch.Tensor):
    """Indices sorting by (value desc, token asc) using a stable library sort."""
    by_tok = torch.sort(tokens, stable=True).indices
    v = values[by_tok]
    idx = torch.sort(v, descending=True, stable=True).indices
    return by_tok[idx]
