"""CPU oracle (test infrastructure, not the product).  See mlpf_oracle.py."""
from .mlpf_oracle import (round_bf16, is_bf16_matrix, quantize_weights, activation, layer_norm, linear,
                          element_types, embed, attention_weights, attention_event,
                          attention_event_tiled, encoder_layer, heads, forward, schedule,
                          parity_metrics, argmax_agreement)
from .candidates import build_candidates
