"""SwiftCache layer-streamed prefill hot path, B200-native."""
